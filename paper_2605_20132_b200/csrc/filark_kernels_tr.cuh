// filark_kernels_tr.cuh -- time-major chunks ([n_t][n_ch], PAPER.md:160 dims='nt_nc'): lanes are CHANNELS,
// warps are TIME SLICES.
//
// The same steps S0..S7, recurrences, tables, carried state, history, control block and work-item protocol
// as filark_push_cm_kernel (filark_kernels.cuh), with the roles of the two axes exchanged:
//
//   * a CTA owns 32 ADJACENT channels; lane l of every warp is channel 32 b + l.  A warp therefore reads and
//     writes 128 contiguous bytes of a time row with one plain 4-byte access per lane: nothing is
//     transposed, nothing goes through shared memory, rows need no alignment;
//   * a tile is 32 slots of L = 24 rows; warp w of 16 owns slots 2w ("lo") and 2w + 1 ("hi") as the two halves
//     of its f32x2 registers, so the zero-state local pass and the fix-up are the code of the channel-major
//     kernel (local_pass, uniform-register table operands);
//   * the scan over the slots is not a scan but a HAND-OFF: warp w waits for a flag in shared memory, takes
//     the state warp w - 1 left for the section, advances it over its own two slots (A^L twice: 8 FMA) and
//     passes it on.  Every warp does the same work, so after the first tile the warps run staggered by one
//     hand-off each and do not wait; warp 0 takes what warp 15 left for the tile before.  The 5-step shuffle
//     scan, the staging of both outputs, the gather moves and every CTA barrier of a transposing kernel are
//     gone ("Time-major").
//
// Work items are (segment of tiles, block of 32 channels), claimed by the CTA; a CTA barrier separates items
// and the chunks of a launch (where raw samples wait for the next chunk), nothing else does.
// Not here: the trigger (the host takes filark_push_cm_kernel<.., kTM = true> when one is set).
#pragma once
#include "filark_kernels.cuh"

namespace filark {

constexpr int kTrL = 24;                                  // rows per slot
constexpr int kTrWarps = 16;
constexpr int kTrRows = 2 * kTrWarps * kTrL;              // 768 rows per tile
constexpr int kTrCh = 32;                                 // channels per CTA
constexpr int kTrRing = kMaxSec + 1;                      // sections + the pair of averages
// dynamic shared memory (floats): the ring [kTrRing][kTrWarps][32] of float2, the waiting raw samples [kTrL][32]
constexpr int kTrRingFloats = kTrRing * kTrWarps * 32 * 2;
constexpr int kTrSmemFloats = kTrRingFloats + kTrL * 32;

// geometry of a chunk for tiles of 32 slots (make_geom of filark_kernels.cuh counts 64)
__device__ __forceinline__ Geom tr_geom(unsigned r0, int n_base, int n_rem)
{
    constexpr int L = kTrL;
    Geom g;
    const int carry = ((int)r0 + n_rem) / L;
    const int n_full = n_base + carry;
    g.r0 = (int)r0;
    g.r1 = (int)r0 + n_rem - carry * L;
    const int slots = n_full + (g.r1 ? 1 : 0);
    g.n_tiles = (slots + 31) / 32;
    g.q_last = n_full - 32 * (g.n_tiles - 1);
    g.vec4 = false;
    return g;
}

// grid <= SM count, block = 16 warps, dynamic shared memory = kTrSmemFloats floats (+ the second history
// buffer, see kTrSmemBytes).  Everything about the control block and the overlap of consecutive launches is
// as in filark_push_cm_kernel.
constexpr size_t kTrSmemBytes = sizeof(float) * (size_t)(kTrSmemFloats + kTrL * 32);

template <int kForm>
__global__ void __launch_bounds__(kTrWarps * 32, 1)
filark_push_tr_kernel(const __grid_constant__ PushParams<kTrL> p)
{
    constexpr int L = kTrL, W = kTrWarps;
    constexpr bool kAllKinds = (kForm & 1) != 0;
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    float2* const ring = reinterpret_cast<float2*>(fk_smem);        // [kTrRing][W][32]: state handed from warp to warp
    float* const hs0 = fk_smem + kTrRingFloats;                       // two buffers [L][32] of raw samples waiting for the
                                                                      // next chunk: chunk k reads buffer k & 1, fills the other
    __shared__ int flag[kTrRing][W];                                  // sequence number of the tile the slot belongs to
    __shared__ unsigned sh_ctl[32];
    __shared__ unsigned sh_flag;
    __shared__ unsigned sh_item;
    __shared__ int sh_tile0[kMaxBatch + 1];
    __shared__ unsigned sh_geo[kMaxBatch];
    if (threadIdx.x < kTrRing * W) (&flag[0][0])[threadIdx.x] = -1;
    if (threadIdx.x == 0) sh_flag = 0u;

    if (p.wait_prior) asm volatile("griddepcontrol.wait;" ::: "memory");

    // ---- control slot of this launch (see filark_push_cm_kernel)
    CmCtl* const cc = p.cctl;
    if (warp == 0) {
        const unsigned* cw = reinterpret_cast<const unsigned*>(cc);
        unsigned v = ld_relaxed(cw + lane);
        const unsigned e = __shfl_sync(0xffffffffu, v, kCtlEpoch);
        const unsigned rp = __shfl_sync(0xffffffffu, v, kCtlSlotWords * (e & 1u) + 7);
        const unsigned need = __shfl_sync(0xffffffffu, v, kCtlSlotWords * (e & 1u) + 4 + rp);
        unsigned ex = __shfl_sync(0xffffffffu, v, kCtlExited + rp);
        const unsigned R0 = __shfl_sync(0xffffffffu, v, kCtlSlotWords * (e & 1u) + 2);
        int carry = 0;
        for (int k0 = 0; k0 < p.n_push; k0 += 32) {
            const int k = k0 + lane;
            int inc = 0;
            unsigned geo = 0;
            if (k < p.n_push) {
                const unsigned r0k = k == 0 ? R0 : (R0 + p.ck[k].t_cum) % (unsigned)L;
                const Geom gk = tr_geom(r0k, p.ck[k].n_base, p.ck[k].n_rem);
                inc = gk.n_tiles;
                geo = r0k | ((unsigned)gk.r1 << 8) | ((unsigned)gk.q_last << 16);
            }
            if (p.n_push > 1) {
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const int u = __shfl_up_sync(0xffffffffu, inc, d);
                    if (lane >= d) inc += u;
                }
            }
            if (k < p.n_push) { sh_tile0[k + 1] = carry + inc; sh_geo[k] = geo; }
            carry += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (lane == 0) sh_tile0[0] = 0;
        while ((int)(ex - need) < 0)                                   // launch e - kCmDepth must have completed
            ex = __shfl_sync(0xffffffffu, ld_relaxed(&cc->exited[rp]), 0);
        sh_ctl[lane] = v;
    }
    __syncthreads();
    const unsigned epoch = sh_ctl[kCtlEpoch];
    const unsigned rpos = sh_ctl[kCtlSlotWords * (epoch & 1u) + 7];
    const unsigned* sl = &sh_ctl[kCtlSlotWords * (epoch & 1u)];
    const unsigned long long seen = (unsigned long long)sl[0] | ((unsigned long long)sl[1] << 32);
    const unsigned seq0 = sl[3];
    const int ns = state_floats(p.n_sec);
    const int n_tiles_all = sh_tile0[p.n_push];
    auto chunk_of = [&](int gt) -> int {
        if (p.n_push == 1) return 0;
        const int a = lane + 1, b = lane + 33;
        const unsigned m0 = __ballot_sync(0xffffffffu, a < p.n_push && sh_tile0[a] <= gt);
        const unsigned m1 = __ballot_sync(0xffffffffu, b < p.n_push && sh_tile0[b] <= gt);
        return __shfl_sync(0xffffffffu, __popc(m0) + __popc(m1), 0);
    };
    auto geom_of = [&](int k) -> Geom {
        const unsigned w = sh_geo[k];
        Geom g;
        g.r0 = (int)(w & 0xffu); g.r1 = (int)((w >> 8) & 0xffu); g.q_last = (int)(w >> 16);
        g.n_tiles = sh_tile0[k + 1] - sh_tile0[k];
        g.vec4 = false;
        return g;
    };
    const int seg_tiles = min(p.seg_tiles, n_tiles_all);
    const int n_seg = seg_tiles == n_tiles_all ? 1 : (n_tiles_all + seg_tiles - 1) / seg_tiles;
    const unsigned n_units = (unsigned)((p.n_ch + kTrCh - 1) / kTrCh);
    const unsigned n_items = (unsigned)n_seg * n_units;

    unsigned pend = 0;
    auto claim_issue = [&]() {
        if (threadIdx.x == 0)
            asm volatile("atom.global.add.u32 %0, [%1], 1;" : "=r"(pend) : "l"(&cc->work[rpos]) : "memory");
    };
    // (thread 0 publishes the claim in sh_item before a CTA barrier, claim_take runs behind it)
    auto claim_take = [&](int& gt, int& gtend, int& seg, int& cb) -> bool {
        const unsigned it = sh_item - sl[8 + rpos];
        if (it >= n_items) return false;
        seg = n_seg == 1 ? 0 : (int)(it / n_units);
        cb = (int)(it - (unsigned)seg * n_units);
        gt = seg * seg_tiles;
        gtend = min(n_tiles_all, gt + seg_tiles);
        return true;
    };

    // ---- hand the control block to the next launch, then let it start
    unsigned tk = 0;
    if (warp == 0 && lane == 0) tk = atomicAdd(&cc->ticket, 1u);
    int gt = 0, gtend = 0, seg = 0, cb = 0;
    claim_issue();
    if (threadIdx.x == 0) sh_item = pend;
    __syncthreads();
    bool have = claim_take(gt, gtend, seg, cb);
    __syncthreads();                                 // (sh_item is rewritten at the item's end)
    claim_issue();
    if (warp == 0) {
        tk = __shfl_sync(0xffffffffu, tk, 0);
        if (lane == 0) {
            if (tk == gridDim.x - 1) {                                // every CTA has read slot[e & 1]
                CmSlot* nx = &cc->slot[(epoch + 1u) & 1u];
                const Chunk& cl = p.ck[p.n_push - 1];
                __stcg(&nx->seen, seen + (unsigned long long)cl.t_cum + (unsigned long long)cl.n_t);
                __stcg(&nx->r0, (sh_geo[p.n_push - 1] >> 8) & 0xffu);
                __stcg(&nx->seq0, seq0 + (unsigned)n_seg);
                for (unsigned j = 0; j < (unsigned)kCmDepth; ++j) {
                    __stcg(&nx->cum[j], sl[4 + j] + (j == rpos ? gridDim.x : 0u));
                    __stcg(&nx->wbase[j], sl[8 + j] + (j == rpos ? n_items + 2u * gridDim.x : 0u));
                }
                __stcg(&nx->ring, rpos + 1u == (unsigned)kCmDepth ? 0u : rpos + 1u);
                __stcg(&cc->ticket, 0u);
                st_release(&cc->epoch, epoch + 1u);
                __threadfence();
            }
            *reinterpret_cast<volatile unsigned*>(&sh_flag) = 1u;
        }
    }
    {
        unsigned f;
        do f = __shfl_sync(0xffffffffu, *reinterpret_cast<volatile unsigned*>(&sh_flag), 0); while (f == 0u);
    }
    asm volatile("griddepcontrol.launch_dependents;");

    const int wp = (warp + W - 1) & (W - 1);         // the warp this one takes the state from
    int seqno = 0;                                    // tiles this CTA has started: the sequence number of the ring
    while (have) {
        const int ch = cb * kTrCh + lane;
        const bool ok = ch < p.n_ch;
        // (lanes of the last block that have no channel compute on a copy of the last channel and store nothing:
        // the block then runs the same unpredicated row code as every other one)
        const int chl = ok ? ch : p.n_ch - 1;
        // ---- the item begins: (segment seg, channels 32 cb ..).  Its carried state goes into the ring as if warp
        // W - 1 had left it for a tile before; the raw samples waiting in front of a chunk go to the history buffer.
        __syncthreads();                             // every warp is done with the item before
        {
            const unsigned need = seq0 + (unsigned)seg;
            unsigned v = ok ? ld_acquire(p.progress + ch) : need;
            while (!__all_sync(0xffffffffu, (int)(v - need) >= 0)) v = ok ? ld_acquire(p.progress + ch) : need;
        }
        int kc = chunk_of(gt);
        Geom g = geom_of(kc);
        int tile = gt - sh_tile0[kc];
        for (int k = warp; k <= p.n_sec; k += W) {
            float2 s = make_float2(0.0f, 0.0f);
            if (ok) {
                const float* gs = p.state + (long long)ch * ns + 2 * k;
                s = make_float2(ld_relaxed_f32(gs), ld_relaxed_f32(gs + 1));
            }
            ring[(k * W + W - 1) * 32 + lane] = s;
            if (lane == 0) flag[k][W - 1] = seqno - 1;
        }
        if (tile == 0)
            for (int e = warp; e < g.r0; e += W)
                hs0[(kc & 1) * L * 32 + e * 32 + lane] = ok ? ld_relaxed_f32(p.hist + (long long)ch * kHist + e) : 0.0f;
        __syncthreads();

        for (; gt < gtend; ++gt, ++seqno, ++tile) {
            if (tile == g.n_tiles) {                 // the item goes on in the next chunk
                ++kc; g = geom_of(kc); tile = 0;
                if (g.r0 != 0) __syncthreads();      // (what waits in front of it was put into the history buffer by a warp of the tile before)
            }
            const Chunk& ck = p.ck[kc];
            const bool item_end = gt + 1 == gtend;
            const int n_t = ck.n_t;
            const int t0 = tile * kTrRows - g.r0;                     // sample of tile position 0
            const int q = tile == g.n_tiles - 1 ? g.q_last : 32;      // full slots of this tile: the state moves over those only
            const int ta = t0 + 2 * L * warp;                         // sample of this warp's first row
            const bool inside = ta >= 0 && ta + 2 * L <= n_t;
            const float* hs_rd = hs0 + (kc & 1) * L * 32;
            float* hs_wr = hs0 + ((kc + 1) & 1) * L * 32;

            // ---- S0: the warp's 2 L rows of its 32 channels
            float2 x[L];
            {
                const float* ip = ck.in + (long long)ta * ck.in_pitch + chl;
                const int pitch = (int)ck.in_pitch;
                if (inside) {
                    // (two running row pointers: one 64-bit multiply-add per access instead of an address built per row)
                    const float* plo = ip;
                    const float* phi = ip + L * pitch;
#pragma unroll
                    for (int i = 0; i < L; ++i) { x[i] = make_float2(__ldcs(plo), __ldcs(phi)); plo += pitch; phi += pitch; }
                } else {
                    // an edge of the chunk: rows in front of it are the samples that waited for it, rows behind it are zero
                    const float* plo = ip;
                    const float* phi = ip + L * pitch;
#pragma unroll
                    for (int i = 0; i < L; ++i) {
                        const int tl = ta + i, th = ta + L + i;
                        float a = 0.0f, b = 0.0f;
                        if (tl < 0) { if (tl + g.r0 >= 0) a = hs_rd[(tl + g.r0) * 32 + lane]; }
                        else if (tl < n_t) a = __ldcs(plo);
                        if (th < 0) { if (th + g.r0 >= 0) b = hs_rd[(th + g.r0) * 32 + lane]; }
                        else if (th < n_t) b = __ldcs(phi);
                        x[i] = make_float2(a, b);
                        plo += pitch; phi += pitch;
                    }
                }
            }
            // the samples of the trailing partial slot wait for whoever continues the channels: the next chunk of
            // this item (history buffer) or the next item / launch (the handle's history rows)
            if (tile == g.n_tiles - 1 && g.r1 != 0 && warp == (q >> 1)) {
                if (item_end) {
                    if (ok) {
                        float* hd = p.hist + (long long)ch * kHist;
#pragma unroll
                        for (int j = 0; j < L; ++j) if (j < g.r1) hd[j] = (q & 1) ? x[j].y : x[j].x;
                    }
                    __threadfence();
                } else {
#pragma unroll
                    for (int j = 0; j < L; ++j) if (j < g.r1) hs_wr[j * 32 + lane] = (q & 1) ? x[j].y : x[j].x;
                }
            }
            {
                const float2 gn = f2(p.gain);
#pragma unroll
                for (int i = 0; i < L; ++i) x[i] = mul2(x[i], gn);
            }
            const int need = warp == 0 ? seqno - 1 : seqno;
            const bool adv_lo = 2 * warp < q, adv_hi = 2 * warp + 1 < q;
            const bool save = item_end && warp == W - 1 && ok;
            float* const gst = p.state + (long long)ch * ns;

            // ---- S1..S3 per section
#pragma unroll 1
            for (int k = 0; k < p.n_sec; ++k) {
                const SecParams<L>& T = p.sec[k];
                float2 s1, s2;
                if (kAllKinds) {
                    switch (T.kind) {
                        case kKindDF2: local_pass<L, kKindDF2>(x, T, s1, s2); break;
                        case kKindDelta: local_pass<L, kKindDelta>(x, T, s1, s2); break;
                        case kKindDeltaG: local_pass<L, kKindDeltaG>(x, T, s1, s2); break;
                        case kKindNormal: local_pass<L, kKindNormal>(x, T, s1, s2); break;
                        default: local_pass<L, kKindDF2G>(x, T, s1, s2); break;
                    }
                } else {
                    if (T.kind == kKindDF2) local_pass<L, kKindDF2>(x, T, s1, s2);
                    else local_pass<L, kKindDelta>(x, T, s1, s2);
                }
                // S2, the hand-off: the state entering this warp's lo slot is what the warp before left
                while (*reinterpret_cast<volatile int*>(&flag[k][wp]) < need) { }
                asm volatile("" ::: "memory");
                const float2 c = ring[(k * W + wp) * 32 + lane];
                const float P0 = T.P[0], P1 = T.P[1], P2 = T.P[2], P3 = T.P[3];
                const float o1 = fmaf(P0, c.x, fmaf(P1, c.y, s1.x)), o2 = fmaf(P2, c.x, fmaf(P3, c.y, s2.x));   // ... its hi slot
                const float n1 = fmaf(P0, o1, fmaf(P1, o2, s1.y)), n2 = fmaf(P2, o1, fmaf(P3, o2, s2.y));       // ... the next warp's lo slot
                const float2 out = adv_hi ? make_float2(n1, n2) : (adv_lo ? make_float2(o1, o2) : c);
                ring[(k * W + warp) * 32 + lane] = out;
                __threadfence_block();
                __syncwarp();
                if (lane == 0) *reinterpret_cast<volatile int*>(&flag[k][warp]) = seqno;
                if (save) __stcg(reinterpret_cast<float2*>(gst + 2 * k), out);
                // S3 fix-up: y[i] += g1[i] s1 + g2[i] s2
                const float2 Ea = make_float2(c.x, o1), Eb = make_float2(c.y, o2);
#pragma unroll
                for (int i = 0; i < L; i += 2) {
                    const float4 gg = *reinterpret_cast<const float4*>(&T.g[i][0]);
                    x[i] = fma2(gg.x, Ea, fma2(gg.y, Eb, x[i]));
                    x[i + 1] = fma2(gg.z, Ea, fma2(gg.w, Eb, x[i + 1]));
                }
            }
            // ---- S7 for the filtered rows
            if (ck.filt) {
                float* fp = ck.filt + (long long)ta * ck.out_pitch + ch;
                const int pitch = (int)ck.out_pitch;
                if (inside && ok) {
                    float* plo = fp;
                    float* phi = fp + L * pitch;
#pragma unroll
                    for (int i = 0; i < L; ++i) { __stcs(plo, x[i].x); __stcs(phi, x[i].y); plo += pitch; phi += pitch; }
                } else if (ok) {
#pragma unroll
                    for (int i = 0; i < L; ++i) {
                        if ((unsigned)(ta + i) < (unsigned)n_t) __stcs(fp + i * pitch, x[i].x);
                        if ((unsigned)(ta + L + i) < (unsigned)n_t) __stcs(fp + (L + i) * pitch, x[i].y);
                    }
                }
            }
            // ---- S4..S6: energy, the two averages, ratio
            const float as = p.avg.alpha[0], al = p.avg.alpha[1];
            float2 sp = make_float2(0.0f, 0.0f), lp = sp;
#pragma unroll
            for (int i = 0; i < L; ++i) {
                const float2 e = mul2(x[i], x[i]);
                x[i] = e;
                sp = fma2(as, sp, e); lp = fma2(al, lp, e);
            }
            const float bLs = p.avg.betaL[0], bLl = p.avg.betaL[1];
            while (*reinterpret_cast<volatile int*>(&flag[p.n_sec][wp]) < need) { }
            asm volatile("" ::: "memory");
            const float2 cm = ring[(p.n_sec * W + wp) * 32 + lane];                       // (sta~, lta~) entering the lo slot
            const float Os = sp.x + fmaf(-bLs, cm.x, cm.x), Ol = lp.x + fmaf(-bLl, cm.y, cm.y);   // ... the hi slot
            const float Ns = sp.y + fmaf(-bLs, Os, Os), Nl = lp.y + fmaf(-bLl, Ol, Ol);
            {
                const float2 out = adv_hi ? make_float2(Ns, Nl) : (adv_lo ? make_float2(Os, Ol) : cm);
                ring[(p.n_sec * W + warp) * 32 + lane] = out;
                __threadfence_block();
                __syncwarp();
                if (lane == 0) *reinterpret_cast<volatile int*>(&flag[p.n_sec][warp]) = seqno;
                if (save) __stcg(reinterpret_cast<float2*>(gst + 2 * p.n_sec), out);
            }
            // the carried state of the item is complete with warp W - 1's last hand-off: tell whoever continues
            if (item_end && warp == W - 1) {
                __threadfence();
                if (ok) st_release(p.progress + ch, seq0 + (unsigned)seg + 1u);
            }
            if (ck.cf) {
                // warm-up (reading R10): samples whose index since create/reset is < lta_len give cf = 0
                const long long rem = (long long)p.lta_len - (long long)(seen + ck.t_cum) - t0;   // first tile position with cf != 0
                const float ratio = p.ratio, thr = p.lta_thr;
                float2 Ps = make_float2(cm.x, Os), Pl = make_float2(cm.y, Ol);
                const bool live = fmaf(-bLl, cm.y, cm.y) > thr && fmaf(-bLl, Ol, Ol) > thr;
                const int base = 2 * L * warp;
                if (rem <= base && __all_sync(0xffffffffu, live)) {
#pragma unroll
                    for (int i = 0; i < L; ++i) {
                        Ps = fma2(as, Ps, x[i]); Pl = fma2(al, Pl, x[i]);
                        const float2 num = mul2(Ps, f2(ratio));
                        x[i] = mul2(num, make_float2(rcp_fast(Pl.x), rcp_fast(Pl.y)));
                    }
                } else {
                    const int wm = rem > (1 << 30) ? (1 << 30) : (rem < 0 ? 0 : (int)rem);
#pragma unroll
                    for (int i = 0; i < L; ++i) {
                        Ps = fma2(as, Ps, x[i]); Pl = fma2(al, Pl, x[i]);
                        const float qa = (Ps.x * ratio) * rcp_fast(Pl.x), qb = (Ps.y * ratio) * rcp_fast(Pl.y);
                        x[i].x = (Pl.x > thr && base + i >= wm) ? qa : 0.0f;
                        x[i].y = (Pl.y > thr && base + L + i >= wm) ? qb : 0.0f;
                    }
                }
                float* cp = ck.cf + (long long)ta * ck.out_pitch + ch;
                const int pitch = (int)ck.out_pitch;
                if (inside && ok) {
                    float* plo = cp;
                    float* phi = cp + L * pitch;
#pragma unroll
                    for (int i = 0; i < L; ++i) { __stcs(plo, x[i].x); __stcs(phi, x[i].y); plo += pitch; phi += pitch; }
                } else if (ok) {
#pragma unroll
                    for (int i = 0; i < L; ++i) {
                        if ((unsigned)(ta + i) < (unsigned)n_t) __stcs(cp + i * pitch, x[i].x);
                        if ((unsigned)(ta + L + i) < (unsigned)n_t) __stcs(cp + (L + i) * pitch, x[i].y);
                    }
                }
            }
        }
        // ---- the next item
        if (threadIdx.x == 0) sh_item = pend;
        __syncthreads();
        have = claim_take(gt, gtend, seg, cb);
        claim_issue();
    }
    // completion: count this CTA out (launch e + kCmDepth waits until all of them are)
    __syncthreads();
    if (threadIdx.x == 0)
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(&cc->exited[rpos]) : "memory");
    // a launch never completes before the launch in front of it
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

}  // namespace filark
