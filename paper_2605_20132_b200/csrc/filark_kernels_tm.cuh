// filark_kernels_tm.cuh -- time-major ([n_t][n_ch], PAPER.md:160 dims='nt_nc') push kernel.
//
// Same steps S0..S7 and the same mathematics as the channel-major kernel (filark_kernels.cuh):
// stream-aligned slots of L samples, zero-state local pass per section, exact block powers for
// the carry, fix-up rows C A^i from the constant bank.  The mapping differs because adjacent
// channels are contiguous here:
//   - a lane owns TWO ADJACENT CHANNELS as the halves of its packed f32x2 registers (one 8-byte
//     load per time sample, a warp reads 256 contiguous bytes of a row: no shared-memory
//     transpose, no staging);
//   - the W warps of a CTA own W consecutive slots of the same 64 channels, so the scan over slots
//     runs ACROSS WARPS: every warp leaves its slot's zero-state end state in shared memory, and
//     after one barrier warp w folds the states of the warps before it,
//     E_w = A^L E_(w-1) + v_(w-1), E_0 = carried state (at most W - 1 dependent steps);
//   - the tiles (W slots x 64 channels) of a push are work items in tile-major order, taken
//     round-robin by the resident CTAs.  Tile t of a 64-channel block needs, for section k, only
//     the state that tile t - 1 of the block left after ITS section k: a per-section look-back.
//     The producer publishes that state (ring of two tiles per block and section) and then a
//     per-(block, section) count of published tiles; the consumer polls the count just before the
//     barrier of its section k.  Consecutive tiles of a block thus run one section apart, on
//     different CTAs, and the number of CTAs at work is not limited by the number of blocks.
//     (A tile depends only on a lower item index and every CTA is resident: the waits end.)
// The raw tail of a push (samples that do not fill a slot) waits in `hist` ([2][kHist][n_ch],
// double-buffered by push parity because different warps read and write it in the same push).
#pragma once
#include "filark_kernels.cuh"

namespace filark {

constexpr int kTmWarps = 8;            // slots per CTA tile
constexpr int kTmL = 16;               // slot length of the time-major kernel

// Extra arguments of the time-major kernel (the tables come with PushParams<kTmL>).
constexpr int kTmStages = kMaxSec + 1;  // sections + the averages
struct TmArgs {
    float* hist2;            // [2][kHist][n_ch]
    float4* carry;           // [n_cb][2][kTmStages][32]: state after a tile's last slot, per stage
    unsigned* published;     // [n_cb][32]: tiles of the running push published, per stage
    int vec2;                // 8-byte accesses are legal (even pitches, 8-byte aligned bases)
};

__device__ __forceinline__ float2 tm_load(const float* __restrict__ row, int c, bool v0, bool v1, bool vec2)
{
    float2 r = make_float2(0.0f, 0.0f);
    if (vec2 && v1) r = __ldcs(reinterpret_cast<const float2*>(row + c));
    else { if (v0) r.x = __ldcs(row + c); if (v1) r.y = __ldcs(row + c + 1); }
    return r;
}
__device__ __forceinline__ void tm_store(float* __restrict__ row, int c, bool v0, bool v1, bool vec2, float2 v)
{
    if (vec2 && v1) __stcs(reinterpret_cast<float2*>(row + c), v);
    else { if (v0) __stcs(row + c, v.x); if (v1) __stcs(row + c + 1, v.y); }
}

// state matvec on channel pairs: (r1, r2) = A (e1, e2) + (v1, v2), A row-major 2x2 (uniform)
__device__ __forceinline__ void tm_step(const float (&P)[4], float2& e1, float2& e2, float2 v1, float2 v2)
{
    const float2 n1 = fma2(P[0], e1, fma2(P[1], e2, v1));
    const float2 n2 = fma2(P[2], e1, fma2(P[3], e2, v2));
    e1 = n1; e2 = n2;
}

template <int L, int W>
__global__ void __launch_bounds__(W * 32, 3)
filark_push_tm_kernel(const __grid_constant__ PushParams<L> p, const __grid_constant__ TmArgs a)
{
    // end states of the W slots: [0], [1] by section parity, [2] the averages (own copy: no barrier
    // separates their reads from the next tile's first section)
    __shared__ float4 vbuf[3][W][32];
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;

    const unsigned r0 = p.ctl->r0, par = p.ctl->pad & 1u;
    const unsigned long long seen = p.ctl->seen;
    const int n_t = p.n_t, n_ch = p.n_ch, n_sec = p.n_sec;
    const long long total = (long long)r0 + n_t;
    const int n_full = (int)(total / L), r1 = (int)(total - (long long)n_full * L);
    const int n_tiles = (n_full + (r1 ? 1 : 0) + W - 1) / W;
    const int n_cb = (n_ch + 63) / 64;
    const float* __restrict__ hrd = a.hist2 + (size_t)par * kHist * n_ch;
    float* __restrict__ hwr = a.hist2 + (size_t)(par ^ 1u) * kHist * n_ch;
    const bool vec2 = a.vec2 != 0, hvec2 = vec2 && (n_ch & 1) == 0;
    const float as = p.avg.alpha[0], al = p.avg.alpha[1];
    const float bLs = p.avg.betaL[0], bLl = p.avg.betaL[1];

    for (unsigned item = blockIdx.x; item < (unsigned)n_tiles * (unsigned)n_cb; item += gridDim.x) {
        const int tile = (int)(item / (unsigned)n_cb), cb = (int)(item - (unsigned)tile * (unsigned)n_cb);
        const int c = cb * 64 + 2 * lane;
        const bool v0 = c < n_ch, v1 = c + 1 < n_ch;
        const int slot = tile * W + warp;
        const int t0 = slot * L - (int)r0;                           // input index of the slot's first sample
        const int q_t = min(max(n_full - tile * W, 0), W);           // full slots in this tile
        const bool last = tile == n_tiles - 1;
        // the warp whose carry-in / carry-out is the state after the tile's last FULL slot
        const bool pub_in = warp == q_t, pub_out = q_t == W && warp == W - 1;
        float4* ring_rd = a.carry + ((size_t)cb * 2 + ((tile + 1) & 1)) * kTmStages * 32;   // written by tile - 1
        float4* ring_wr = a.carry + ((size_t)cb * 2 + (tile & 1)) * kTmStages * 32;
        unsigned* pubs = a.published + (size_t)cb * 32;

        // state entering the tile, stage k: tile 0 from the handle's state ([word][n_ch]), later
        // tiles from the ring once tile - 1 has published stage k (warp 0 polled before the barrier)
        auto wait_stage = [&](int k) {
            if (tile > 0 && warp == 0) {
                unsigned done;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(done) : "l"(pubs + k) : "memory");
                    done = __shfl_sync(0xffffffffu, done, 0);
                } while (done < (unsigned)tile);
            }
        };
        auto carry_in = [&](int k) -> float4 {
            float4 v;
            if (tile == 0) {
                const float* s1 = p.state + (size_t)(2 * k) * n_ch, *s2 = s1 + n_ch;
                v.x = v0 ? __ldcg(s1 + c) : 0.0f; v.y = v1 ? __ldcg(s1 + c + 1) : 0.0f;
                v.z = v0 ? __ldcg(s2 + c) : 0.0f; v.w = v1 ? __ldcg(s2 + c + 1) : 0.0f;
            } else {
                v = __ldcg(ring_rd + k * 32 + lane);
            }
            return v;
        };
        // the state after the tile's last full slot: to the ring (+ count) for tile + 1, or, on the
        // last tile, to the handle's state (and the count back to 0 for the next push)
        auto carry_out = [&](int k, float4 v) {
            if (last) {
                float* s1 = p.state + (size_t)(2 * k) * n_ch, *s2 = s1 + n_ch;
                if (v0) { s1[c] = v.x; s2[c] = v.z; }
                if (v1) { s1[c + 1] = v.y; s2[c + 1] = v.w; }
                if (lane == 0) pubs[k] = 0u;
            } else {
                ring_wr[k * 32 + lane] = v;
                __threadfence();
                __syncwarp();
                if (lane == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(pubs + k), "r"((unsigned)(tile + 1)) : "memory");
            }
        };

        // ---- S0: load (history for t < 0, zeros for t >= n_t) ----------------------------------
        float2 x[L];
        const bool inside = t0 >= 0 && t0 + L <= n_t;                // the slot lies inside the push (uniform)
        if (inside) {
            const float* row = p.in + (size_t)t0 * p.in_pitch;
#pragma unroll
            for (int i = 0; i < L; ++i) x[i] = tm_load(row + (size_t)i * p.in_pitch, c, v0, v1, vec2);
        } else {
#pragma unroll
            for (int i = 0; i < L; ++i) {
                const int t = t0 + i;
                float2 v = make_float2(0.0f, 0.0f);
                if (t < 0) v = tm_load(hrd + (size_t)((int)r0 + t) * n_ch, c, v0, v1, hvec2);
                else if (t < n_t) v = tm_load(p.in + (size_t)t * p.in_pitch, c, v0, v1, vec2);
                x[i] = v;
            }
        }
        if (slot == n_full && r1 != 0) {
            // the trailing partial slot: its raw samples wait for the next push
#pragma unroll
            for (int i = 0; i < L; ++i)
                if (i < r1) tm_store(hwr + (size_t)i * n_ch, c, v0, v1, hvec2, x[i]);
        }
        {
            const float2 gn = f2(p.gain);
#pragma unroll
            for (int i = 0; i < L; ++i) x[i] = mul2(x[i], gn);
        }
        // ---- S1..S3 per section -----------------------------------------------------------------
        for (int k = 0; k < n_sec; ++k) {
            const SecParams<L>& T = p.sec[k];
            float2 s1, s2;
            switch (T.kind) {
                case kKindDF2: local_pass<L, kKindDF2>(x, T, s1, s2); break;
                case kKindDelta: local_pass<L, kKindDelta>(x, T, s1, s2); break;
                case kKindDeltaG: local_pass<L, kKindDeltaG>(x, T, s1, s2); break;
                case kKindNormal: local_pass<L, kKindNormal>(x, T, s1, s2); break;
                default: local_pass<L, kKindDF2G>(x, T, s1, s2); break;
            }
            vbuf[k & 1][warp][lane] = make_float4(s1.x, s1.y, s2.x, s2.y);
            wait_stage(k);
            __syncthreads();
            const float4 S = carry_in(k);
            float2 e1 = make_float2(S.x, S.y), e2 = make_float2(S.z, S.w);
            for (int j = 0; j < warp; ++j) {
                const float4 v = vbuf[k & 1][j][lane];
                tm_step(T.P, e1, e2, make_float2(v.x, v.y), make_float2(v.z, v.w));
            }
            if (pub_in) carry_out(k, make_float4(e1.x, e1.y, e2.x, e2.y));
            if (pub_out) {
                float2 n1 = e1, n2 = e2;
                tm_step(T.P, n1, n2, s1, s2);
                carry_out(k, make_float4(n1.x, n1.y, n2.x, n2.y));
            }
#pragma unroll
            for (int i = 0; i < L; ++i) x[i] = fma2(T.g[i][0], e1, fma2(T.g[i][1], e2, x[i]));
        }
        if (p.filt) {
            if (inside) {
                float* row = p.filt + (size_t)t0 * p.out_pitch;
#pragma unroll
                for (int i = 0; i < L; ++i) tm_store(row + (size_t)i * p.out_pitch, c, v0, v1, vec2, x[i]);
            } else {
#pragma unroll
                for (int i = 0; i < L; ++i) {
                    const int t = t0 + i;
                    if (t >= 0 && t < n_t) tm_store(p.filt + (size_t)t * p.out_pitch, c, v0, v1, vec2, x[i]);
                }
            }
        }
        // ---- S4..S6: energy, the two averages, ratio --------------------------------------------
        float2 sp = make_float2(0.0f, 0.0f), lp = sp;
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const float2 e = mul2(x[i], x[i]);
            x[i] = e;
            sp = fma2(as, sp, e); lp = fma2(al, lp, e);
        }
        vbuf[2][warp][lane] = make_float4(sp.x, sp.y, lp.x, lp.y);
        wait_stage(n_sec);
        __syncthreads();
        const float4 M = carry_in(n_sec);
        float2 es = make_float2(M.x, M.y), el = make_float2(M.z, M.w);
        for (int j = 0; j < warp; ++j) {
            const float4 v = vbuf[2][j][lane];
            es = add2(make_float2(v.x, v.y), fma2(-bLs, es, es));        // alpha^L e + v
            el = add2(make_float2(v.z, v.w), fma2(-bLl, el, el));
        }
        if (pub_in) carry_out(n_sec, make_float4(es.x, es.y, el.x, el.y));
        if (pub_out) {
            const float2 ns = add2(sp, fma2(-bLs, es, es)), nl = add2(lp, fma2(-bLl, el, el));
            carry_out(n_sec, make_float4(ns.x, ns.y, nl.x, nl.y));
        }
        if (p.cf) {
            // warm-up (reading R10) and division guard (R11), per sample
            const long long rem = (long long)p.lta_len - (long long)seen - t0;   // first i with cf != 0
            const int wm = rem > (1 << 30) ? (1 << 30) : (rem < 0 ? 0 : (int)rem);
            const float ratio = p.ratio, thr = p.lta_thr;
#pragma unroll
            for (int i = 0; i < L; ++i) {
                es = fma2(as, es, x[i]); el = fma2(al, el, x[i]);
                const float qa = (es.x * ratio) * rcp_fast(el.x), qb = (es.y * ratio) * rcp_fast(el.y);
                float2 o;
                o.x = (el.x > thr && i >= wm) ? qa : 0.0f;
                o.y = (el.y > thr && i >= wm) ? qb : 0.0f;
                const int t = t0 + i;
                if (inside || (t >= 0 && t < n_t)) tm_store(p.cf + (size_t)t * p.out_pitch, c, v0, v1, vec2, o);
            }
        }
    }

    // the last CTA to finish advances the control block
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned t = atomicAdd(&p.ctl->ticket, 1u);
        if (t == gridDim.x - 1) {
            p.ctl->r0 = (unsigned)r1;
            p.ctl->seen = seen + (unsigned long long)n_t;
            p.ctl->pad = par ^ 1u;
            p.ctl->ticket = 0u;
            __threadfence();
        }
    }
}

}  // namespace filark
