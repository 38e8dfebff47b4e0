// filark_kernels.cuh -- sm_100a kernels of the fused SOS + STA/LTA stream path.
//
// Steps (include/filark_stream.h): S0 load, S1 per-section local scan,
// S2 warp-shuffle combine, S3 fix-up + carried state, S4 energy, S5 STA/LTA scans,
// S6 ratio + warm-up, S7 store.  One launch per push; the chunk is read once from HBM and
// each output is written once.
//
// Channel-major mapping (time contiguous): one warp owns one channel at a time.  The time axis
// of a push is cut into sub-blocks of L samples ("slots"); a tile is 64 consecutive slots and
// lane l owns slots 2l ("lo") and 2l+1 ("hi"), i.e. 2L contiguous samples, in registers through
// every section and the STA/LTA.  The two slots of a lane are two independent recurrence chains
// interleaved in program order (B200 issues FFMA2 at the cost of two FFMA, so plain scalar FFMA
// on two chains is as fast and needs no register pairing -- DESIGN.md 6).  Tiles of a channel
// are processed in time order by the same warp; the carried state sits in shared memory between
// tiles and in global memory between pushes.
//
// Persistent grid: one CTA per SM, W warps per CTA; warp (b, w) walks the channels
// b + grid (w + W i), i = 0, 1, ...  While a tile is computed, the next tile (of the same or of
// the warp's next channel) and that channel's carried state are already in flight into the
// warp's second shared-memory buffer (cp.async, 16 B per lane, zero-filled outside the push).
//
// Ragged pushes need no second code path: slots are aligned to the END of the push, the first
// slot is the short one (r <= L samples, zero-padded at its front -- a zero-state recurrence
// stays at rest through leading zeros), and it always sits in the hi slot of lane 0 of tile 0
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

constexpr int kMaxSec = 16;
constexpr int kMaxWarps = 16;          // warps per CTA (one CTA per SM)
constexpr int kSteps = 5;              // log2(32) scan steps
constexpr int kKindDF2 = 0, kKindDF2G = 1, kKindDelta = 2, kKindDeltaG = 3, kKindNormal = 4;

// ---- device table of one sub-block length L (floats); see build_variant_table() ----------------
// per section, stride SecTab<L>::stride:
//   [0] kind (int bits)  [1..5] local-pass coefficients  [7] scan steps needed (int bits)
//   [8..11]  P = A^L                       [12..31] Q[d] = A^(2L 2^d), d = 0..4 (row-major 2x2)
//   G0: 2L rows (g1, g2): rows -L..-1 are zero, row i >= 0 is C A^i     (+ 4 floats pad)
//   G1: the same shifted down by one row (row j holds G0 row j-1): 16-byte aligned odd shifts
// after the sections, the averages block (kAvgFloats):
//   [0] alpha_s [1] alpha_l  [2..3] 1 - alpha^L  [4..13] 1 - alpha^(2L 2^d) (s,l interleaved)
//   [14] 1/N_s [15] 1/N_l
// What depends on the push (the length r of its first slot) travels in PushParams.
template <int L> struct SecTab {
    static constexpr int g0 = 32;
    static constexpr int gsz = 4 * L + 4;
    static constexpr int g1 = g0 + gsz;
    static constexpr int stride = g1 + gsz;
};
constexpr int kOffKind = 0, kOffCoef = 1, kOffNSteps = 7, kOffP = 8, kOffQ = 12;
constexpr int kAvgBetaL = 2, kAvgBetaQ = 4, kAvgInvN = 14, kAvgFloats = 16;

// Carried state of one channel (floats): [0, 2 n_sec) section states, then sta~, lta~, the
// number of samples seen since create/reset (uint32 bits, saturating), one pad word.
__host__ __device__ constexpr int state_floats(int n_sec) { return 2 * n_sec + 4; }
constexpr unsigned kSeenMax = 0x7fffffffu;    // >= any lta_len; only ever moved as bits

struct PushParams {
    const float* in;
    float* filt;
    float* cf;
    const float* tab;        // table of the chosen L (device)
    float* state;            // channel-major: [n_ch][state_floats]; time-major kernels: [state_floats][n_ch]
    long long n_t, in_pitch, out_pitch;
    int n_ch, n_sec;
    int n_tiles;             // tiles per channel
    int lead;                // idle slots in front of the first one (0, or 1 when r < L)
    int r;                   // samples in the first slot, 1..L
    int pad0;                // zeros in front of sample 0: lead L + (L - r)
    int last_lane, last_half;// lane / half of the slot holding the last sample (in the last tile)
    int lta_len;
    int vec4;                // 16-byte global accesses are legal (alignment, pitch, n_t % 4 == 0)
    float gain, ratio, lta_thr;
    float beta_r[2];         // 1 - alpha^r            (sta, lta): carry across the first slot
    float inv_sh[2];         // alpha^-(L - r)         (sta, lta): second pass of the first slot
    float apow_r[kMaxSec][4];// A^r per section, row-major 2x2
};

// ---- small PTX wrappers ------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16(float* dst, const float* src, int src_bytes)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async4(float* dst, const float* src, int src_bytes)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(s), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void st_stream(float* p, float v) { __stcs(p, v); }
__device__ __forceinline__ void st_stream4(float* p, float4 v) { __stcs(reinterpret_cast<float4*>(p), v); }
__device__ __forceinline__ float rcp_fast(float a) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }

template <int L> struct Geo {
    static constexpr int pitch = 2 * L + 4;        // floats per lane region: LDS.128 conflict-free
    static constexpr int tile = 64 * L;            // samples per tile
    static constexpr int buf_floats = 32 * pitch;
    static constexpr int chunks = L / 2;           // 16-byte chunks per lane region
};

// All dynamic shared memory, addressed by float offsets so that every access is provably a
// shared-memory access (32-bit addresses, LDS/STS instead of generic LD/ST).
extern __shared__ __align__(16) float fk_smem[];

// Shared memory of one warp: two tile buffers (input of tile k / staging of its outputs, and the
// prefetched input of tile k+1) and two copies of the channel state.
constexpr int kStateSmem = 40;                     // >= state_floats(kMaxSec), multiple of 4
template <int L> __host__ __device__ constexpr int warp_smem_floats() { return 2 * Geo<L>::buf_floats + 2 * kStateSmem; }

// S0: start the asynchronous copy of one tile of one channel into `buf` (padded lane regions:
// tile-local sample e lives at buf[e + 4 (e / 2L)]) and of the channel's carried state into
// `wst`.  t0 = time index (within the push) of the tile's position 0; samples outside [0, n_t)
// are zero-filled.
template <int L>
__device__ __forceinline__ void issue_tile_load(const PushParams& p, int ch, int tile, int buf, int wst,
                                                int lane, bool with_state)
{
    const int t0 = tile * Geo<L>::tile - p.pad0;
    const int n_t = (int)p.n_t;
    const float* __restrict__ src = p.in + (long long)ch * p.in_pitch;
    if (p.vec4) {
        // valid 16-byte chunks of this tile: [c_lo, c_hi)
        const int c_lo = t0 < 0 ? (-t0 >> 2) : 0;
        const int c_hi = min(Geo<L>::tile, n_t - t0) >> 2;
        const unsigned span = (unsigned)(c_hi - c_lo);
        const float* __restrict__ srct = src + t0;
#pragma unroll
        for (int m = 0; m < Geo<L>::chunks; ++m) {
            const int c = 32 * m + lane;
            const bool ok = (unsigned)(c - c_lo) < span;
            cp_async16(&fk_smem[buf + 4 * c + 4 * (c / Geo<L>::chunks)], ok ? srct + 4 * c : src, ok ? 16 : 0);
        }
    } else {
#pragma unroll 8
        for (int m = 0; m < 2 * L; ++m) {
            const int e = 32 * m + lane;
            const int t = t0 + e;
            const bool ok = (unsigned)t < (unsigned)n_t;
            cp_async4(&fk_smem[buf + e + 4 * (e / (2 * L))], ok ? src + t : src, ok ? 4 : 0);
        }
    }
    if (with_state) {
        const int ns = state_floats(p.n_sec);
        const float* gst = p.state + (long long)ch * ns;
        if (lane < ns) cp_async4(&fk_smem[wst + lane], gst + lane, 4);
        if (lane + 32 < ns) cp_async4(&fk_smem[wst + lane + 32], gst + lane + 32, 4);
    }
    cp_async_commit();
}

// S7: the lane regions of `buf` -> one output array (coalesced 16-byte stores).
template <int L>
__device__ __forceinline__ void store_tile(const PushParams& p, float* __restrict__ dst, int buf, int lane, int t0)
{
    const int n_t = (int)p.n_t;
    if (p.vec4) {
        const int c_lo = t0 < 0 ? (-t0 >> 2) : 0;
        const int c_hi = min(Geo<L>::tile, n_t - t0) >> 2;
        const unsigned span = (unsigned)(c_hi - c_lo);
        float* __restrict__ dstt = dst + t0;
#pragma unroll
        for (int m = 0; m < Geo<L>::chunks; ++m) {
            const int c = 32 * m + lane;
            const float4 v = *reinterpret_cast<const float4*>(&fk_smem[buf + 4 * c + 4 * (c / Geo<L>::chunks)]);
            if ((unsigned)(c - c_lo) < span) st_stream4(dstt + 4 * c, v);
        }
    } else {
#pragma unroll 8
        for (int m = 0; m < 2 * L; ++m) {
            const int e = 32 * m + lane;
            const int t = t0 + e;
            const float v = fk_smem[buf + e + 4 * (e / (2 * L))];
            if ((unsigned)t < (unsigned)n_t) st_stream(dst + t, v);
        }
    }
}

template <int L>
__device__ __forceinline__ void regs_to_buf(const float (&lo)[L], const float (&hi)[L], int buf, int lane)
{
    float4* d = reinterpret_cast<float4*>(&fk_smem[buf + lane * Geo<L>::pitch]);
#pragma unroll
    for (int q = 0; q < L / 4; ++q) {
        d[q] = make_float4(lo[4 * q], lo[4 * q + 1], lo[4 * q + 2], lo[4 * q + 3]);
        d[L / 4 + q] = make_float4(hi[4 * q], hi[4 * q + 1], hi[4 * q + 2], hi[4 * q + 3]);
    }
}

// S1: zero-state response of one section on the lane's two slots; returns their end states.
template <int L, int KIND>
__device__ __forceinline__ void local_pass(float (&lo)[L], float (&hi)[L], int Toff,
                                           float& a1, float& a2, float& b1, float& b2)
{
    const float* T = &fk_smem[Toff];
    const float c0 = T[kOffCoef], c1 = T[kOffCoef + 1], c2 = T[kOffCoef + 2], c3 = T[kOffCoef + 3];
    a1 = a2 = b1 = b2 = 0.0f;                       // (a1, a2): state of the lo slot, (b1, b2): hi slot
    if (KIND == kKindDF2) {
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const float wa = fmaf(c0, a1, fmaf(c1, a2, lo[i]));
            const float wb = fmaf(c0, b1, fmaf(c1, b2, hi[i]));
            lo[i] = fmaf(c2, a1, fmaf(c3, a2, wa));
            hi[i] = fmaf(c2, b1, fmaf(c3, b2, wb));
            a2 = a1; a1 = wa; b2 = b1; b1 = wb;
        }
    } else if (KIND == kKindDelta) {
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const float ua = fmaf(c0, a1, fmaf(c1, a2, lo[i]));
            const float ub = fmaf(c0, b1, fmaf(c1, b2, hi[i]));
            lo[i] = fmaf(c2, a1, ua);
            hi[i] = fmaf(c2, b1, ub);
            a2 += ua; a1 = ua; b2 += ub; b1 = ub;
        }
    } else if (KIND == kKindDeltaG) {
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const float ua = fmaf(c0, a1, fmaf(c1, a2, lo[i]));
            const float ub = fmaf(c0, b1, fmaf(c1, b2, hi[i]));
            lo[i] = fmaf(c3, a2, fmaf(c2, a1, ua));
            hi[i] = fmaf(c3, b2, fmaf(c2, b1, ub));
            a2 += ua; a1 = ua; b2 += ub; b1 = ub;
        }
    } else if (KIND == kKindNormal) {
        const float nc1 = -c1;
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const float xa = lo[i], xb = hi[i];
            lo[i] = fmaf(c2, a1, fmaf(c3, a2, xa));
            hi[i] = fmaf(c2, b1, fmaf(c3, b2, xb));
            const float na = fmaf(c0, a1, fmaf(c1, a2, xa));
            const float nb = fmaf(c0, b1, fmaf(c1, b2, xb));
            a2 = fmaf(c0, a2, nc1 * a1); b2 = fmaf(c0, b2, nc1 * b1);
            a1 = na; b1 = nb;
        }
    } else {                                        // kKindDF2G: explicit b0 = coefficient 4
        const float c4 = T[kOffCoef + 4];
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const float wa = fmaf(c0, a1, fmaf(c1, a2, lo[i]));
            const float wb = fmaf(c0, b1, fmaf(c1, b2, hi[i]));
            lo[i] = fmaf(c2, a1, fmaf(c3, a2, c4 * wa));
            hi[i] = fmaf(c2, b1, fmaf(c3, b2, c4 * wb));
            a2 = a1; a1 = wa; b2 = b1; b1 = wb;
        }
    }
}

// One tile of one channel, samples already in lo/hi: S1..S7.  `buf` stages the outputs.
// stab / buf / wst are float offsets into fk_smem.
template <int L>
__device__ __forceinline__ void process_tile(const PushParams& p, int stab, int buf, int wst, float (&lo)[L],
                                             float (&hi)[L], int ch, int tile, int lane, unsigned seen)
{
    using ST = SecTab<L>;
    const bool first = tile == 0, last = tile == p.n_tiles - 1;
    const int t0 = tile * Geo<L>::tile - p.pad0;
    const bool inj_hi = first && p.lead != 0;   // carried state enters the hi slot of lane 0 (ragged tile 0)
    const int r = first ? p.r : L;              // samples in the slot that receives the carried state
    const int sh = L - r;
    const int jl = last ? p.last_lane : 31;     // lane of the slot holding the tile's last sample
    const bool out_hi = last ? p.last_half != 0 : true;
    const float m_lo = (lane == 0 && !inj_hi) ? 1.0f : 0.0f;
    const float m_hi = (lane == 0 && inj_hi) ? 1.0f : 0.0f;
    // per-lane fix-up table offset (floats) inside a section's table: lane 0's injected slot is
    // short by sh samples, so its rows are shifted down by sh
    int goff = ST::g0 + 2 * L;
    if (lane == 0 && sh != 0) goff = (sh & 1) ? ST::g1 + 2 * (L - sh + 1) : ST::g0 + 2 * (L - sh);

    // ---- S1..S3 per section -------------------------------------------------------------------
    for (int k = 0; k < p.n_sec; ++k) {
        const int To = stab + k * ST::stride;
        const int kind = __float_as_int(fk_smem[To + kOffKind]);
        float a1, a2, b1, b2;
        switch (kind) {
            case kKindDF2: local_pass<L, kKindDF2>(lo, hi, To, a1, a2, b1, b2); break;
            case kKindDelta: local_pass<L, kKindDelta>(lo, hi, To, a1, a2, b1, b2); break;
            case kKindDeltaG: local_pass<L, kKindDeltaG>(lo, hi, To, a1, a2, b1, b2); break;
            case kKindNormal: local_pass<L, kKindNormal>(lo, hi, To, a1, a2, b1, b2); break;
            default: local_pass<L, kKindDF2G>(lo, hi, To, a1, a2, b1, b2); break;
        }
        // S2: carried state S into its slot, then an inclusive scan of the lane totals
        const float2 S = *reinterpret_cast<const float2*>(&fk_smem[wst + 2 * k]);
        const float4 Pm = *reinterpret_cast<const float4*>(&fk_smem[To + kOffP]);     // A^L
        const float4 Ar = *reinterpret_cast<const float4*>(&p.apow_r[k][0]);          // A^r (first slot)
        const float4 Au = first ? Ar : Pm;
        const float i1 = fmaf(Au.x, S.x, Au.y * S.y), i2 = fmaf(Au.z, S.x, Au.w * S.y);
        a1 = fmaf(m_lo, i1, a1); a2 = fmaf(m_lo, i2, a2);                             // state after the lo slot
        b1 = fmaf(m_hi, i1, b1); b2 = fmaf(m_hi, i2, b2);
        float W1 = fmaf(Pm.x, a1, fmaf(Pm.y, a2, b1)), W2 = fmaf(Pm.z, a1, fmaf(Pm.w, a2, b2));
        const int nsteps = __float_as_int(fk_smem[To + kOffNSteps]);
#pragma unroll
        for (int d = 0; d < kSteps; ++d) {
            if (d < nsteps) {
                const float4 Q = *reinterpret_cast<const float4*>(&fk_smem[To + kOffQ + 4 * d]);
                float U1 = __shfl_up_sync(0xffffffffu, W1, 1 << d), U2 = __shfl_up_sync(0xffffffffu, W2, 1 << d);
                const bool act = lane >= (1 << d);
                U1 = act ? U1 : 0.0f; U2 = act ? U2 : 0.0f;
                W1 = fmaf(Q.x, U1, fmaf(Q.y, U2, W1));
                W2 = fmaf(Q.z, U1, fmaf(Q.w, U2, W2));
            }
        }
        float E1 = __shfl_up_sync(0xffffffffu, W1, 1), E2 = __shfl_up_sync(0xffffffffu, W2, 1);
        E1 = lane == 0 ? 0.0f : E1; E2 = lane == 0 ? 0.0f : E2;    // state entering the lane's lo slot
        // carry-in of the hi slot: P E + (state after lo from rest)
        float o1 = fmaf(Pm.x, E1, fmaf(Pm.y, E2, a1)), o2 = fmaf(Pm.z, E1, fmaf(Pm.w, E2, a2));
        // new carried state: state after the slot holding the last sample
        const float n1 = __shfl_sync(0xffffffffu, out_hi ? W1 : o1, jl);
        const float n2 = __shfl_sync(0xffffffffu, out_hi ? W2 : o2, jl);
        if (lane == 0) {
            *reinterpret_cast<float2*>(&fk_smem[wst + 2 * k]) = make_float2(n1, n2);
            if (inj_hi) { o1 = S.x; o2 = S.y; } else { E1 = S.x; E2 = S.y; }
        }
        // S3 fix-up: y[i] += g1[i] s1 + g2[i] s2
        const float4* G = reinterpret_cast<const float4*>(&fk_smem[To + goff]);
#pragma unroll
        for (int i = 0; i < L; i += 2) {
            const float4 gg = G[i >> 1];
            lo[i] = fmaf(gg.x, E1, fmaf(gg.y, E2, lo[i]));
            hi[i] = fmaf(gg.x, o1, fmaf(gg.y, o2, hi[i]));
            lo[i + 1] = fmaf(gg.z, E1, fmaf(gg.w, E2, lo[i + 1]));
            hi[i + 1] = fmaf(gg.z, o1, fmaf(gg.w, o2, hi[i + 1]));
        }
    }

    if (p.filt) {
        regs_to_buf<L>(lo, hi, buf, lane);
        __syncwarp();
        store_tile<L>(p, p.filt + (long long)ch * p.out_pitch, buf, lane, t0);
        __syncwarp();
    }

    // ---- S4..S6: energy, the two averages, ratio --------------------------------------------
    const int AV = stab + p.n_sec * ST::stride;
    const float as = fk_smem[AV], al = fk_smem[AV + 1];
    float sa = 0.0f, la = 0.0f, sb = 0.0f, lb = 0.0f;       // (sta, lta) x (lo slot, hi slot) from rest
#pragma unroll
    for (int i = 0; i < L; ++i) {
        const float ea = lo[i] * lo[i], eb = hi[i] * hi[i];
        lo[i] = ea; hi[i] = eb;
        sa = fmaf(as, sa, ea); la = fmaf(al, la, ea);
        sb = fmaf(as, sb, eb); lb = fmaf(al, lb, eb);
    }
    const int ks = wst + 2 * p.n_sec;
    const float2 M = *reinterpret_cast<const float2*>(&fk_smem[ks]);           // carried (sta~, lta~)
    // carried averages into their slot: + alpha^len M = M - (1 - alpha^len) M
    const float bLs = fk_smem[AV + kAvgBetaL], bLl = fk_smem[AV + kAvgBetaL + 1];
    const float brs = first ? p.beta_r[0] : bLs, brl = first ? p.beta_r[1] : bLl;
    const float is = fmaf(-brs, M.x, M.x), il = fmaf(-brl, M.y, M.y);
    sa = fmaf(m_lo, is, sa); la = fmaf(m_lo, il, la);
    sb = fmaf(m_hi, is, sb); lb = fmaf(m_hi, il, lb);
    float Ws = sb + fmaf(-bLs, sa, sa), Wl = lb + fmaf(-bLl, la, la);          // alpha^L lo + hi
#pragma unroll
    for (int d = 0; d < kSteps; ++d) {
        const float2 q = *reinterpret_cast<const float2*>(&fk_smem[AV + kAvgBetaQ + 2 * d]);
        float Us = __shfl_up_sync(0xffffffffu, Ws, 1 << d), Ul = __shfl_up_sync(0xffffffffu, Wl, 1 << d);
        const bool act = lane >= (1 << d);
        Us = act ? Us : 0.0f; Ul = act ? Ul : 0.0f;
        Ws += fmaf(-q.x, Us, Us); Wl += fmaf(-q.y, Ul, Ul);
    }
    float Es = __shfl_up_sync(0xffffffffu, Ws, 1), El = __shfl_up_sync(0xffffffffu, Wl, 1);
    Es = lane == 0 ? 0.0f : Es; El = lane == 0 ? 0.0f : El;
    float Os = sa + fmaf(-bLs, Es, Es), Ol = la + fmaf(-bLl, El, El);          // carry-in of the hi slot
    const float Ns = __shfl_sync(0xffffffffu, out_hi ? Ws : Os, jl);
    const float Nl = __shfl_sync(0xffffffffu, out_hi ? Wl : Ol, jl);
    if (lane == 0) {
        *reinterpret_cast<float2*>(&fk_smem[ks]) = make_float2(Ns, Nl);
        // the short slot starts its second pass sh zeros early: M alpha^-sh decays to M on them
        const float Mvs = first ? M.x * p.inv_sh[0] : M.x, Mvl = first ? M.y * p.inv_sh[1] : M.y;
        if (inj_hi) { Os = Mvs; Ol = Mvl; } else { Es = Mvs; El = Mvl; }
    }

    if (p.cf) {
        // warm-up (reading R10): samples whose index since create/reset is < lta_len give cf = 0
        const long long rem = (long long)p.lta_len - (long long)seen - t0;     // first tile position with cf != 0
        const float ratio = p.ratio, thr = p.lta_thr;
        // l~ never drops below alpha^L times its carry-in inside a slot (e >= 0); the idle slot in
        // front of a ragged push (lo slot of lane 0) holds no sample
        const bool live = (fmaf(-bLl, El, El) > thr || (lane == 0 && inj_hi)) && fmaf(-bLl, Ol, Ol) > thr;
        if (rem <= 0 && __all_sync(0xffffffffu, live)) {
#pragma unroll
            for (int i = 0; i < L; ++i) {
                Es = fmaf(as, Es, lo[i]); El = fmaf(al, El, lo[i]);
                Os = fmaf(as, Os, hi[i]); Ol = fmaf(al, Ol, hi[i]);
                lo[i] = (Es * ratio) * rcp_fast(El);
                hi[i] = (Os * ratio) * rcp_fast(Ol);
            }
        } else {
            const int wm = rem > (1 << 30) ? (1 << 30) : (rem < 0 ? 0 : (int)rem);
            const int base = 2 * lane * L;
#pragma unroll
            for (int i = 0; i < L; ++i) {
                Es = fmaf(as, Es, lo[i]); El = fmaf(al, El, lo[i]);
                Os = fmaf(as, Os, hi[i]); Ol = fmaf(al, Ol, hi[i]);
                const float qa = (Es * ratio) * rcp_fast(El), qb = (Os * ratio) * rcp_fast(Ol);
                lo[i] = (El > thr && base + i >= wm) ? qa : 0.0f;
                hi[i] = (Ol > thr && base + L + i >= wm) ? qb : 0.0f;
            }
        }
        regs_to_buf<L>(lo, hi, buf, lane);
        __syncwarp();
        store_tile<L>(p, p.cf + (long long)ch * p.out_pitch, buf, lane, t0);
    }
    __syncwarp();
}

// Warps per CTA the register file allows (one CTA per SM): 128 / 168 / 255 registers per thread.
template <int L> __host__ __device__ constexpr int cm_max_warps() { return L <= 24 ? 16 : (L <= 32 ? 12 : 8); }

// Channel-major push: grid <= SM count, block = W * 32 (W <= cm_max_warps<L>()); dynamic shared memory =
// table + W * warp_smem_floats<L>() floats.
template <int L>
__global__ void __launch_bounds__(cm_max_warps<L>() * 32, 1)
filark_push_cm_kernel(const __grid_constant__ PushParams p)
{
    const int tab_floats = p.n_sec * SecTab<L>::stride + kAvgFloats;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;
    const int wbase = tab_floats + warp * warp_smem_floats<L>();      // two tile buffers, then two state copies
    const int wst0 = wbase + 2 * Geo<L>::buf_floats;

    // warp (b, w) walks the channels b + grid (w + W i)
    const int stride = gridDim.x * W;
    int ch = blockIdx.x + gridDim.x * warp, tile = 0, cur = 0, wcur = 0;
    if (ch < p.n_ch) issue_tile_load<L>(p, ch, 0, wbase, wst0, lane, true);
    for (int i = threadIdx.x; i < tab_floats / 4; i += blockDim.x)
        reinterpret_cast<float4*>(fk_smem)[i] = __ldg(reinterpret_cast<const float4*>(p.tab) + i);
    __syncthreads();

    const int ns = state_floats(p.n_sec);
    unsigned seen = 0;
    while (ch < p.n_ch) {
        int nch = ch, ntile = tile + 1;
        if (ntile == p.n_tiles) { ntile = 0; nch = ch + stride; }
        const int buf = wbase + cur * Geo<L>::buf_floats;
        const int wst = wst0 + wcur * kStateSmem;
        cp_async_wait_all();
        __syncwarp();
        float lo[L], hi[L];
        {
            const float4* s = reinterpret_cast<const float4*>(&fk_smem[buf + lane * Geo<L>::pitch]);
            const float gn = p.gain;
#pragma unroll
            for (int q = 0; q < L / 4; ++q) {
                const float4 a = s[q], b = s[L / 4 + q];
                lo[4 * q] = a.x * gn; lo[4 * q + 1] = a.y * gn; lo[4 * q + 2] = a.z * gn; lo[4 * q + 3] = a.w * gn;
                hi[4 * q] = b.x * gn; hi[4 * q + 1] = b.y * gn; hi[4 * q + 2] = b.z * gn; hi[4 * q + 3] = b.w * gn;
            }
        }
        if (tile == 0) seen = __float_as_uint(fk_smem[wst + ns - 2]);
        __syncwarp();
        if (nch < p.n_ch)
            issue_tile_load<L>(p, nch, ntile, wbase + (cur ^ 1) * Geo<L>::buf_floats,
                               wst0 + (wcur ^ 1) * kStateSmem, lane, ntile == 0);
        process_tile<L>(p, 0, buf, wst, lo, hi, ch, tile, lane, seen);
        if (ntile == 0) {
            // channel done: carried state and sample count back to global memory
            if (lane == 0) {
                const unsigned long long s2 = (unsigned long long)seen + (unsigned long long)p.n_t;
                fk_smem[wst + ns - 2] = __uint_as_float(s2 > kSeenMax ? kSeenMax : (unsigned)s2);
            }
            __syncwarp();
            float* gst = p.state + (long long)ch * ns;
            if (lane < ns) gst[lane] = fk_smem[wst + lane];
            if (lane + 32 < ns) gst[lane + 32] = fk_smem[wst + lane + 32];
            wcur ^= 1;
        }
        ch = nch; tile = ntile; cur ^= 1;
    }
}

// Diagnostic kernel (FILARK_FLAG_SERIAL_SCAN; also the time-major path for now): one thread per
// channel, serial in time, the same state-space sections and the same state contents, no blocked
// scan.  Element (c, t) of a chunk is at c * sc + t * st; state word i of channel c is at
// c * state_sc + i * state_sk.  tab = table of any L (only the coefficients and 1/N are read).
__global__ void __launch_bounds__(128)
filark_push_serial_kernel(const __grid_constant__ PushParams p, int sec_stride, long long sc_in,
                          long long st_in, long long sc_out, long long st_out, long long state_sc,
                          long long state_sk)
{
    __shared__ float coef[kMaxSec][8];
    __shared__ float cinv[2];
    for (int i = threadIdx.x; i < p.n_sec * 8; i += blockDim.x)
        coef[i >> 3][i & 7] = p.tab[(i >> 3) * sec_stride + (i & 7)];
    if (threadIdx.x < 2) cinv[threadIdx.x] = p.tab[p.n_sec * sec_stride + kAvgInvN + threadIdx.x];
    __syncthreads();
    const int ch = blockIdx.x * blockDim.x + threadIdx.x;
    if (ch < p.n_ch) {
        float s[2 * kMaxSec + 2];
        const int nf = 2 * p.n_sec + 2;
        for (int i = 0; i < nf; ++i) s[i] = p.state[ch * state_sc + i * state_sk];
        const unsigned seen = __float_as_uint(p.state[ch * state_sc + nf * state_sk]);
        const float cs = cinv[0], cl = cinv[1];
        float ms = s[nf - 2], ml = s[nf - 1];
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
                    (ml > p.lta_thr && (unsigned long long)seen + (unsigned long long)t >= (unsigned long long)p.lta_len)
                        ? p.ratio * __fdividef(ms, ml) : 0.0f;
        }
        s[nf - 2] = ms; s[nf - 1] = ml;
        for (int i = 0; i < nf; ++i) p.state[ch * state_sc + i * state_sk] = s[i];
        const unsigned long long s2 = (unsigned long long)seen + (unsigned long long)p.n_t;
        p.state[ch * state_sc + nf * state_sk] = __uint_as_float(s2 > kSeenMax ? kSeenMax : (unsigned)s2);
    }
}

}  // namespace filark
