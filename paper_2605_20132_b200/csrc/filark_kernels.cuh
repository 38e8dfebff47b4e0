// filark_kernels.cuh -- sm_100a kernels of the fused SOS + STA/LTA stream path.
//
// Steps (include/filark_stream.h): S0 load, S1 per-section local scan,
// S2 warp-shuffle combine, S3 fix-up + carried state, S4 energy, S5 STA/LTA scans,
// S6 ratio + warm-up, S7 store.  One launch per push; the chunk is read once from HBM and
// each output is written once.
//
// Channel-major mapping (time contiguous): one warp owns one channel at a time.  The time axis
// is cut into sub-blocks of L samples ("slots"); a tile is 64 consecutive slots and lane l owns
// slots 2l ("lo") and 2l+1 ("hi"), i.e. 2L contiguous samples, as the two halves of L packed
// f32x2 registers that stay in registers through every section and the STA/LTA.  Every
// per-sample instruction is an FFMA2 whose third operand -- a section coefficient, a fix-up row
// C A^i, an averaging constant -- is warp-uniform and comes from the kernel-parameter constant
// bank through a uniform register: an FFMA2 with three register-file operands is limited to
// about 2/3 of the FMA pipe by register-file bandwidth on B200, with a uniform operand it runs
// at ~95 % (profiles/).
//
// Slots are aligned to the STREAM, not to the push: the carried state of a channel always
// belongs to a slot boundary.  The samples of a push that do not fill a slot (r1 < L of them)
// are filtered and written like all others (zero-padded slot, outputs of the padding dropped),
// but the state is not advanced over them; their raw values are kept in the handle (`hist`)
// and the next push starts with them (r0 = r1 positions of its first tile come from `hist`,
// their outputs are recomputed and dropped).  Every slot that advances the state is therefore
// full, every lane uses the same fix-up rows, and ragged pushes need no second code path.
// r0 and the sample counter live in device memory (`CmCtl`), so a push has no host-side mutable
// argument and can be replayed from a CUDA graph.
//
// Persistent grid, 16 warps per SM (four small CTAs, or one for long pushes): a warp walks work
// items (segment of tiles, channel).  While a tile is computed, the next tile (of the same or of
// the warp's next channel) and that channel's carried state are already in flight into the
// warp's second shared-memory buffer (cp.async, 16 B per lane, zero-filled outside the push).
// Consecutive pushes of a handle overlap on the device (see filark_push_cm_kernel).  Time-major
// chunks ([n_t][n_ch]) go through the same kernel with a transpose in shared memory (kTM).
//
// The recurrences are exact restatements of the oracle's definition:
//   section:  s[n] = A s[n-1] + B x[n],  y[n] = C s[n-1] + D x[n]           (design.hpp)
//   slot with carry-in s_in, local pass from zero state giving y_loc and end state v:
//             y[i] = y_loc[i] + (C A^i) s_in,   s_out = A^L s_in + v
//   averages: m~[n] = alpha m~[n-1] + e[n]  (m~ = m * N),  cf = (N_l/N_s) s~/l~
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace filark {

constexpr int kMaxSec = 16;
constexpr int kMaxWarps = 16;          // warps per SM
constexpr int kSteps = 5;              // log2(32) scan steps
constexpr int kHist = 64;              // floats of raw history per channel (>= largest L)
constexpr int kKindDF2 = 0, kKindDF2G = 1, kKindDelta = 2, kKindDeltaG = 3, kKindNormal = 4;

// Device-resident control block of a handle.  Consecutive pushes of a handle overlap on the device
// (programmatic dependent launch, see filark_push_cm_kernel), so what a push needs to know about
// its predecessors is double-buffered by push parity: push number e (since create/reset) reads
// slot[e & 1]; the last of its CTAs to have read it writes slot[(e + 1) & 1] and publishes
// epoch = e + 1 before the grid lets its dependents launch.
constexpr int kCmDepth = 3;        // pushes of a handle in flight at most
struct CmSlot {                // 12 words
    unsigned long long seen;   // samples pushed before this push
    unsigned int r0;           // samples waiting in `hist`
    unsigned int seq0;         // segments completed per channel before this push (cumulative, wraps)
    unsigned int cum[kCmDepth];    // CTAs launched by the earlier pushes of ring position j (cumulative, wraps)
    unsigned int ring;         // this push's position in the ring of kCmDepth pushes in flight (kept here, not
                               // taken as epoch % kCmDepth: 2^32 is not a multiple of 3)
    unsigned int wbase[kCmDepth];  // value of work[j] at which the next push of ring position j starts claiming
    unsigned int pad;
};
struct CmCtl {
    CmSlot slot[2];            // words 0..11, 12..23
    unsigned int epoch;        // word 24: pushes started since create/reset
    unsigned int ticket;       // word 25: CTAs of the starting push that have read their slot
    unsigned int exited[kCmDepth];   // words 26..28: CTAs finished, by ring position (cumulative): push
                               // e - kCmDepth and all before it are complete when exited[ring] has
                               // reached slot[e & 1].cum[ring]
    unsigned int work[kCmDepth];     // words 29..31: work items claimed, by ring position (cumulative, never
                               // reset: push e claims work[ring] - slot[e & 1].wbase[ring]), see "Work items"
};
constexpr int kCtlSlotWords = 12, kCtlEpoch = 24, kCtlExited = 26;
static_assert(sizeof(CmSlot) == 4 * kCtlSlotWords && sizeof(CmCtl) == 128, "the control block is read by one warp in one access");

// One SOS section for sub-block length L; every member is warp-uniform and is read straight
// from the constant bank.  Q[d] = A^(2L 2^d); g[i] = C A^i.
template <int L> struct alignas(16) SecParams {
    int kind, nsteps;
    float c[5];
    float pad;
    float P[4];                // A^L, row-major 2x2
    float Q[kSteps][4];
    float g[L][2];
};

// The two exponential averages (index 0: STA, 1: LTA).  beta = 1 - alpha^n keeps full relative
// precision for alpha next to 1; v alpha^n is evaluated as v - beta v.
struct AvgParams {
    float alpha[2];
    float betaL[2];            // 1 - alpha^L
    float betaQ[kSteps][2];    // 1 - alpha^(2L 2^d)
    float invN[2];
};

// Carried state of one channel (floats): [0, 2 n_sec) section states, then sta~, lta~, the
// number of samples seen (serial kernel only; uint32 bits, saturating), then the trigger state
// (kTrigWords words: on/off, peak, t_on as two words; see trigger_tile).
// (padded to a multiple of four words: the state moves in 16-byte pieces)
constexpr int kTrigWords = 4;
__host__ __device__ constexpr int trig_word(int n_sec) { return 2 * n_sec + 3; }
__host__ __device__ constexpr int state_floats(int n_sec) { return (2 * n_sec + 3 + kTrigWords + 3) & ~3; }
constexpr unsigned kSeenMax = 0x7fffffffu;

// One chunk of a launch.  A launch covers up to kMaxBatch consecutive chunks of the stream (one
// for filark_stream_push, the chunks of a filark_stream_push_many schedule otherwise): every
// channel's tiles run through all of them with the carried state staying in shared memory, so
// that a chunk boundary inside a launch costs no hand-over through global memory at all.
// Every member is warp-uniform and is read straight from the parameter bank.
constexpr int kMaxBatch = 64;
struct Chunk {
    const float* in;
    float* filt;
    float* cf;
    long long in_pitch, out_pitch;
    int n_t, n_base, n_rem;  // n_t = n_base L + n_rem
    unsigned t_cum;          // samples of the launch in front of this chunk
};

// One closed event of the on/off trigger (== filark_event_t of include/filark_stream.h).
struct Event {
    long long t_on, t_off;   // sample indices since create/reset: first sample with cf >= thr_on, first later one with cf < thr_off
    int channel;
    float peak;              // largest cf in [t_on, t_off)
};
static_assert(sizeof(Event) == 24, "event record");

template <int L> struct PushParams {
    float* state;            // [n_ch][state_floats]
    float* hist;             // [n_ch][kHist]
    CmCtl* cctl;
    unsigned* progress;      // [n_ch] segments completed per channel since create/reset (cumulative, wraps)
    int n_ch, n_sec, lta_len;
    int n_push;              // chunks of this launch, 1 .. kMaxBatch
    int seg_tiles;           // tiles per work item (host heuristic: about 8 items per resident warp)
    int vec4;                // host's view of the alignment (channel-major: introspection only, the kernel derives
                             // the shift of every row itself, see "Alignment"; time-major: 16-byte stores allowed)
    int wait_prior;          // wait for everything before this launch in the stream before touching memory
    float gain, ratio, lta_thr;
    // trigger on the characteristic function (trigger_tile): off when thr_on <= 0
    float thr_on, thr_off;
    Event* events;           // [ev_cap] closed events, in no particular order
    unsigned* n_events;      // events closed so far (may exceed ev_cap: the excess is dropped and counted)
    unsigned ev_cap;
    AvgParams avg;
    SecParams<L> sec[kMaxSec];
    Chunk ck[kMaxBatch];
};

// Per-push geometry, derived on the device from the control block (host mirror: filark_debug_push_geometry).
struct Geom {
    int r0;                  // tile-space positions [0, r0) of tile 0 come from hist
    int n_tiles;
    int q_last;              // full slots in the last tile, 0..64
    int r1;                  // samples of the trailing partial slot, 0..L-1
    bool vec4;
};
// n_t = n_base L + n_rem is split on the host, so that the device needs no division (every CTA
// of every push derives the geometry in its prologue, a serial chain of scalar instructions).
template <int L>
__host__ __device__ inline Geom make_geom(unsigned r0, int n_base, int n_rem, bool vec4)
{
    Geom g;
    // (r0 < kHist is the tail of the previous push, which may have used a longer L; n_rem < L)
    const int carry = ((int)r0 + n_rem) / L;               // small numerator, compile-time divisor
    const int n_full = n_base + carry;                     // full slots of r0 + n_t samples
    g.r0 = (int)r0;
    g.r1 = (int)r0 + n_rem - carry * L;
    const int slots = n_full + (g.r1 ? 1 : 0);
    g.n_tiles = (slots + 63) >> 6;
    g.q_last = n_full - 64 * (g.n_tiles - 1);
    g.vec4 = vec4 && (r0 & 3u) == 0;
    return g;
}
template <int L>
__host__ __device__ inline Geom make_geom(unsigned r0, int n_t, bool vec4) { return make_geom<L>(r0, n_t / L, n_t % L, vec4); }

// ---- small PTX wrappers ------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16(int dst_off, const float* src, int src_bytes);
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void st_stream(float* p, float v) { __stcs(p, v); }
__device__ __forceinline__ void st_stream4(float* p, float4 v) { __stcs(reinterpret_cast<float4*>(p), v); }
__device__ __forceinline__ float rcp_fast(float a) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
__device__ __forceinline__ unsigned ld_acquire(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// `progress`: the FIRST look at a word (asked for early, where the warp has other latency to sit out) is an
// acquire load at gpu scope; if its value already suffices -- the usual case -- nothing more is needed.
// Otherwise the warp polls with relaxed loads (served by L2, no fence behind them) and ends with one more
// acquire load.  Everything these guard (state, hist) was written before a release at gpu scope and is read
// with loads that bypass L1 (cp.async.cg, ld.relaxed.gpu) issued after the acquire has returned.  The
// control block is read with relaxed loads: its slots are complete before the grid can launch (below).
__device__ __forceinline__ unsigned ld_relaxed(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// (guarded data read with plain instructions: volatile + memory clobber, so that the compiler cannot
// move the load above the poll that guards it -- the __ldcg intrinsic is a pure asm and may be)
__device__ __forceinline__ float ld_relaxed_f32(const float* p)
{
    float v;
    asm volatile("ld.relaxed.gpu.global.f32 %0, [%1];" : "=f"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(unsigned* p, unsigned v)
{
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ float2 f2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 fma2(float a, float2 b, float2 c) { return __ffma2_rn(make_float2(a, a), b, c); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }

template <int L> struct Geo {
    static constexpr int pitch = 2 * L + 4;        // floats per lane region: LDS.128 conflict-free
    static constexpr int tile = 64 * L;            // samples per tile
    static constexpr int buf_floats = 32 * pitch + 4;  // + one chunk: a shifted tile (below) ends in "region 32"
    static constexpr int chunks = L / 2;           // 16-byte chunks per lane region
};

// All dynamic shared memory, addressed by float offsets so that every access is provably a
// shared-memory access (32-bit addresses, LDS/STS instead of generic LD/ST).
extern __shared__ __align__(16) float fk_smem[];

__device__ __forceinline__ void cp_async16(int dst_off, const float* src, int src_bytes)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(&fk_smem[dst_off]);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async4(int dst_off, const float* src, int src_bytes)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(&fk_smem[dst_off]);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(s), "l"(src), "r"(src_bytes) : "memory");
}

// Shared-space accesses by 32-bit address (the carried state of a section is read and written once per
// section: through `fk_smem[...]` the compiler rebuilds the generic-to-shared window address every time)
__device__ __forceinline__ unsigned smem_addr(int float_off) { return (unsigned)__cvta_generic_to_shared(&fk_smem[float_off]); }
__device__ __forceinline__ float2 lds_f2(unsigned sa)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(sa) : "memory");
    return v;
}
__device__ __forceinline__ void sts_f2(unsigned sa, float2 v)
{
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(sa), "f"(v.x), "f"(v.y) : "memory");
}

// Shared memory of one warp: two tile buffers (input of tile k / staging of its outputs, and the
// prefetched input of tile k+1) and two copies of the channel state.
constexpr int kStateSmem = 44;                     // >= state_floats(kMaxSec), multiple of 4
constexpr int kHistSmem = 48;                      // raw history of the next item's channel (r0 < 48)
template <int L> __host__ __device__ constexpr int warp_smem_floats() { return 2 * Geo<L>::buf_floats + 2 * kStateSmem + kHistSmem; }

// Alignment.  Global rows start anywhere (4-byte aligned pointers, any pitch, any n_t) and tile
// position e of a push is input sample t = e - r0 (+ tile offset), so in general neither the row
// nor the tile is 16-byte aligned.  The tile is therefore held in shared memory SHIFTED by
// s = (row address / 4 - r0) mod 4 floats: "raw" position p = e + s has the same alignment as the
// global element it holds, 16-byte chunks of the row are copied to 16-byte chunks of the buffer
// (cp.async 16 B in, STG.128 out; only the at most three elements at either end of a row move one
// by one), and the shift is undone where the lane regions meet the registers (scalar LDS/STS
// instead of 128-bit ones when s != 0).  Input, filt and cf rows each have their own shift.
__device__ __forceinline__ int row_shift(const float* row, int r0)
{
    return (int)(((unsigned)((uintptr_t)row >> 2) - (unsigned)r0) & 3u);
}
// index in a tile buffer of raw position p (padded lane regions)
template <int L> __device__ __forceinline__ int raw_index(int p) { return p + 4 * (p / (2 * L)); }

// Where chunk c = 32 m + lane of a tile (16 bytes, chunks in time order: what one warp instruction moves
// between global and shared memory) sits in a tile buffer with padded lane regions: float offset
// 4 c + 4 (c / C), C = chunks per lane region.  Written as (per-lane base) + (constant of m), so that the
// unrolled copy loops address with immediates and no per-chunk arithmetic: for C | 32 the quotient
// splits at once; for C = 12 (L = 24) c / 12 = lane / 12 + 2 m + (8 m + lane mod 12) / 12, and the last
// term is (2 m) / 3 plus a step at lane mod 12 >= 4 (m mod 3 = 1) or >= 8 (m mod 3 = 2): three bases.
template <int L> struct TimeOrder {
    static constexpr int C = Geo<L>::chunks;
    static_assert(32 % C == 0 || C == 12, "sub-block lengths 8, 16, 24 (and 32, 64)");
    int b0, b1, b2;
    __device__ __forceinline__ explicit TimeOrder(int lane)
    {
        if (C == 12) {
            const int a = lane / 12, r = lane - 12 * a;
            b0 = 4 * lane + 4 * a; b1 = b0 + (r >= 4 ? 4 : 0); b2 = b0 + (r >= 8 ? 4 : 0);
        } else {
            b0 = b1 = b2 = 4 * lane + 4 * (lane / C);
        }
    }
    // (m is a compile-time constant wherever this is used: fully unrolled loops)
    __device__ __forceinline__ int at(int m) const
    {
        if (C == 12) return (m % 3 == 0 ? b0 : (m % 3 == 1 ? b1 : b2)) + 136 * m + 4 * ((2 * m) / 3);
        return b0 + 128 * m + 4 * ((32 * m) / C);
    }
};

// (out of line: the unrolled copies of the shifted path are long, and the kernel's aligned paths are
// faster the smaller the kernel is -- inlined they cost the aligned headline 3 %)
template <int L>
__device__ __noinline__ void issue_tile_input_shifted(const float* __restrict__ src, int n_t, int t0, int s, int buf, int lane,
                                                      const TimeOrder<L> to)
{
    const int tf0 = t0 + 4 * lane - s;
    const float* __restrict__ srct = src + tf0;
#pragma unroll
    for (int m = 0; m <= Geo<L>::chunks; ++m) {
        const int tf = tf0 + 128 * m;
        const int rem = n_t - tf;
        const int bytes = tf < 0 ? 0 : (rem >= 4 ? 16 : (rem > 0 ? 4 * rem : 0));
        if (m == 0) {
            if (tf <= -4 || tf >= 0) {
                cp_async16(buf + to.at(0), srct, bytes);
            } else {
                for (int j = 1; j < 4; ++j) {
                    const int t = tf + j;
                    if (t >= 0) cp_async4(buf + to.at(0) + j, src + (t < n_t ? t : 0), t < n_t ? 4 : 0);
                }
            }
        } else if (m < Geo<L>::chunks || lane == 0) {
            cp_async16(buf + to.at(m), srct + 128 * m, bytes);
        }
    }
}

// S0: start the asynchronous copy of one tile of one channel into `buf` (padded lane regions:
// tile-local sample e lives at buf[e + 4 (e / 2L)]) and, with the channel's first tile, of its
// carried state into `wst`.  Tile-space position e of tile `tile` is input sample
// t = tile 64L + e - r0; t < 0 reads hist[ch][r0 + t], t >= n_t is zero-filled.
// kShift: built for launches with rows that are not 16-byte aligned (the host knows: p.vec4 = 0): their tiles
// take the unrolled shifted paths; otherwise a compact loop serves the rare shifted tile (a handle whose
// sample count is not a multiple of four when an aligned launch arrives) and the kernel stays small.
template <int L, bool kInterior, bool kShift>
__device__ __forceinline__ void issue_tile_input(const PushParams<L>& p, const Chunk& ck, const Geom& g, int ch, int tile, int buf, int lane,
                                                 const TimeOrder<L>& to)
{
    const int t0 = tile * Geo<L>::tile - g.r0;
    const int n_t = ck.n_t;
    const float* __restrict__ src = ck.in + (long long)ch * ck.in_pitch;
    const int s = row_shift(src, g.r0);
    if (kInterior && s == 0 && t0 >= 0 && t0 + Geo<L>::tile <= n_t) {   // aligned interior tile: no bounds
        // (only in the kernel built for long pushes: elsewhere the instruction cache is the scarcer
        // resource and one path serves interior and edge tiles)
        const float* __restrict__ srct = src + t0 + 4 * lane;
#pragma unroll
        for (int m = 0; m < Geo<L>::chunks; ++m) {
            const int c = 32 * m + lane;
            cp_async16(buf + to.at(m), srct + 128 * m, 16);
        }
    } else if (s == 0 && ((g.r0 | n_t) & 3) == 0) {                  // aligned rows, whole chunks only
        // chunk c = 32 m + lane exists if lo <= c < hi (before it: history; behind it: nothing).  Every
        // chunk is copied, the ones that do not exist with src-size 0 (zero fill, nothing is read): what
        // waits in the history is put over the zeros when the tile is taken up.  The bounds are taken
        // relative to the lane once, so that a chunk costs a compare against a constant, a select and the
        // copy, and there is no lane-dependent branch -- this path runs for every tile of an ordinary push.
        // (r0 < 128: only the first 32 chunks can hold history.)
        const int lo = (-t0 >> 2) - lane, hi = ((n_t - t0) >> 2) - lane;
        const float* __restrict__ srct = src + t0 + 4 * lane;
#pragma unroll
        for (int m = 0; m < Geo<L>::chunks; ++m) {
            const bool ok = m == 0 ? (lo <= 0 && 0 < hi) : 32 * m < hi;
            cp_async16(buf + to.at(m), srct + 128 * m, ok ? 16 : 0);
        }
    } else {
        // Shifted rows.  Raw chunk c = 32 m + lane holds input samples tf .. tf + 3, tf = t0 + 4 c - s (16-byte
        // aligned in global memory by the choice of s); one chunk more than a tile has (c = 32 chunks: lane 0
        // only; what it loads beyond the tile is not used).  Chunks before the row (history, put over them when
        // the tile is taken up) or behind it are zero-filled with src-size 0, the chunk that holds the row's
        // end is copied up to there; unrolled with immediate addresses like the aligned path.  Only the chunk
        // that straddles t = 0 (first tile of a chunk, m = 0) moves element by element.
        if constexpr (kShift) {
            issue_tile_input_shifted<L>(src, n_t, t0, s, buf, lane, to);
        } else {
            // raw chunk c holds input samples tf .. tf + 3; samples before the row (t < 0) are history
            // (issue_tile_carry), samples behind it (t >= n_t) are zero-filled; one chunk more than a
            // tile has, because of the shift (what it loads beyond the tile is not used)
    #pragma unroll 1
            for (int c = lane; c <= 32 * Geo<L>::chunks; c += 32) {
                const int tf = t0 + 4 * c - s;
                const int d = buf + 4 * c + 4 * (c / Geo<L>::chunks);
                if (tf >= 0) {
                    const int rem = n_t - tf;
                    const int bytes = rem >= 4 ? 16 : (rem > 0 ? 4 * rem : 0);
                    cp_async16(d, bytes ? src + tf : p.hist, bytes);
                } else if (tf > -4) {
                    for (int j = 1; j < 4; ++j) {
                        const int t = tf + j;
                        if (t >= 0) cp_async4(d + j, src + (t < n_t ? t : 0), t < n_t ? 4 : 0);
                    }
                }
            }
        }
    }
    cp_async_commit();
}

// S0, what the channel carries into its tile 0: the r0 raw samples waiting in `hist` (tile-space
// positions [0, r0)) and the carried state into `wst`.  Both are rewritten by pushes that overlap
// this one on the device: never read through L1, and only after `progress` says they are there.
template <int L>
__device__ __forceinline__ void issue_tile_carry(const PushParams<L>& p, const Geom& g, int ch, int whs, int wst, int lane)
{
    // (history goes to the warp's scratch first: where it belongs in the tile buffer depends on the
    // row's shift, and it is moved there when the tile is taken up)
    const float* __restrict__ hist = p.hist + (long long)ch * kHist;
    if (4 * lane < g.r0) cp_async16(whs + 4 * lane, hist + 4 * lane, 16);
    const int ns = state_floats(p.n_sec);
    const float* gst = p.state + (long long)ch * ns;
    if (4 * lane < ns) cp_async16(wst + 4 * lane, gst + 4 * lane, 16);
    cp_async_commit();
}

template <int L>
__device__ __noinline__ void store_tile_shifted(float* __restrict__ dst, int n_t, int t0, int s, int buf, int lane, const TimeOrder<L> to)
{
    const int e0 = 4 * lane - s, tf0 = t0 + e0;
    float* __restrict__ dstt = dst + tf0;
#pragma unroll
    for (int m = 0; m <= Geo<L>::chunks; ++m) {
        const int e = e0 + 128 * m, tf = tf0 + 128 * m;
        const bool full = e >= 0 && e + 4 <= Geo<L>::tile && tf >= 0 && tf + 4 <= n_t && (m < Geo<L>::chunks || lane == 0);
        if (m < Geo<L>::chunks || lane == 0) {
            const float4 v = *reinterpret_cast<const float4*>(&fk_smem[buf + to.at(m)]);
            if (full) st_stream4(dstt + 128 * m, v);
        }
    }
    const int cand[4] = {0, 32 * Geo<L>::chunks, (s - t0) >> 2, (n_t - t0 + s) >> 2};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int c = cand[i];
        if (c >= 0 && c <= 32 * Geo<L>::chunks && (c & 31) == lane) {
            const int e = 4 * c - s, tf = t0 + e;
            const int b = buf + 4 * c + 4 * (c / Geo<L>::chunks);
            if (!(e >= 0 && e + 4 <= Geo<L>::tile && tf >= 0 && tf + 4 <= n_t)) {
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if ((unsigned)(e + j) < (unsigned)Geo<L>::tile && (unsigned)(tf + j) < (unsigned)n_t)
                        st_stream(dst + tf + j, fk_smem[b + j]);
            }
        }
    }
}

// S7: the lane regions of `buf` -> one output array (coalesced 16-byte stores).  Positions that
// map to t < 0 (recomputed history) or t >= n_t (padding) are dropped.
template <int L, bool kInterior, bool kShift>
__device__ __forceinline__ void store_tile(const Chunk& ck, const Geom& g, float* __restrict__ dst, int buf,
                                           int lane, int t0, int s, const TimeOrder<L>& to)
{
    const int n_t = ck.n_t;
    if (kInterior && s == 0 && t0 >= 0 && t0 + Geo<L>::tile <= n_t) {
        float* __restrict__ dstt = dst + t0 + 4 * lane;
#pragma unroll
        for (int m = 0; m < Geo<L>::chunks; ++m) {
            const int c = 32 * m + lane;
            const float4 v = *reinterpret_cast<const float4*>(&fk_smem[buf + to.at(m)]);
            st_stream4(dstt + 128 * m, v);
        }
    } else if (s == 0 && ((g.r0 | n_t) & 3) == 0) {                  // aligned rows, whole chunks only
        const int lo = (-t0 >> 2) - lane, hi = ((n_t - t0) >> 2) - lane;       // as in issue_tile_input
        float* __restrict__ dstt = dst + t0 + 4 * lane;
#pragma unroll
        for (int m = 0; m < Geo<L>::chunks; ++m) {
            const float4 v = *reinterpret_cast<const float4*>(&fk_smem[buf + to.at(m)]);
            const bool ok = m == 0 ? (lo <= 0 && 0 < hi) : 32 * m < hi;
            if (ok) st_stream4(dstt + 128 * m, v);
        }
    } else {
        // Shifted rows.  Element j of raw chunk c = 32 m + lane is tile position e = 4 c + j - s: only
        // 0 <= e < tile belongs to this tile (the first chunk starts with the previous tile's last samples,
        // the extra chunk ends with the next tile's first ones), and only 0 <= t < n_t exists.  Chunks that lie
        // completely inside go out with one predicated 16-byte store each (unrolled, immediate addresses);
        // the at most four chunks that cross a boundary (e = 0, e = tile, t = 0, t = n_t) follow element by element.
        if constexpr (kShift) {
            store_tile_shifted<L>(dst, n_t, t0, s, buf, lane, to);
        } else {
            // element j of raw chunk c is tile position e = 4 c + j - s: only 0 <= e < tile belongs to
            // this tile (the first chunk starts with the previous tile's last samples, the extra chunk
            // ends with the next tile's first ones), and only 0 <= t < n_t exists
    #pragma unroll 1
            for (int c = lane; c <= 32 * Geo<L>::chunks; c += 32) {
                const int e = 4 * c - s;
                const int tf = t0 + e;
                const float4 v = *reinterpret_cast<const float4*>(&fk_smem[buf + 4 * c + 4 * (c / Geo<L>::chunks)]);
                if (e >= 0 && e + 4 <= Geo<L>::tile && tf >= 0 && tf + 4 <= n_t) {
                    st_stream4(dst + tf, v);
                } else {
                    const float vv[4] = {v.x, v.y, v.z, v.w};
    #pragma unroll
                    for (int j = 0; j < 4; ++j)
                        if ((unsigned)(e + j) < (unsigned)Geo<L>::tile && (unsigned)(tf + j) < (unsigned)n_t)
                            st_stream(dst + tf + j, vv[j]);
                }
            }
        }
    }
}

// Unpack the lane's pairs into its shared-memory region: lo samples then hi samples (raw positions
// 2L lane + s ...: the last few hi samples of a shifted tile fall into the next region).
template <int L>
__device__ __forceinline__ void regs_to_buf(const float2 (&x)[L], int buf, int lane, int s)
{
    if (s == 0) {
        float4* d = reinterpret_cast<float4*>(&fk_smem[buf + lane * Geo<L>::pitch]);
#pragma unroll
        for (int q = 0; q < L / 4; ++q) {
            d[q] = make_float4(x[4 * q].x, x[4 * q + 1].x, x[4 * q + 2].x, x[4 * q + 3].x);
            d[L / 4 + q] = make_float4(x[4 * q].y, x[4 * q + 1].y, x[4 * q + 2].y, x[4 * q + 3].y);
        }
    } else {
        const int base = buf + lane * Geo<L>::pitch + s;
#pragma unroll
        for (int i = 0; i < L; ++i) {
            fk_smem[base + i] = x[i].x;
            const int o = L + i;
            fk_smem[base + o + ((i >= L - 3 && s + o >= 2 * L) ? 4 : 0)] = x[i].y;
        }
    }
}

// The reverse: the lane's region -> packed pairs, times the cascade's gain.
template <int L>
__device__ __forceinline__ void buf_to_regs(float2 (&x)[L], int buf, int lane, int s, float gn)
{
    if (s == 0) {
        const float4* r = reinterpret_cast<const float4*>(&fk_smem[buf + lane * Geo<L>::pitch]);
#pragma unroll
        for (int q = 0; q < L / 4; ++q) {
            const float4 a = r[q], b = r[L / 4 + q];
            x[4 * q] = make_float2(a.x * gn, b.x * gn); x[4 * q + 1] = make_float2(a.y * gn, b.y * gn);
            x[4 * q + 2] = make_float2(a.z * gn, b.z * gn); x[4 * q + 3] = make_float2(a.w * gn, b.w * gn);
        }
    } else {
        const int base = buf + lane * Geo<L>::pitch + s;
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const int o = L + i;
            x[i] = make_float2(fk_smem[base + i] * gn,
                               fk_smem[base + o + ((i >= L - 3 && s + o >= 2 * L) ? 4 : 0)] * gn);
        }
    }
}

// ---- time-major chunks ([n_t][n_ch], PAPER.md:160 dims='nt_nc') --------------------------------
// The same kernel serves them through a transpose in shared memory: a CTA of kTmChannels warps
// owns kTmChannels ADJACENT channels (one per warp, exactly as in the channel-major mapping), and
// its threads move a tile together: thread (c, j) = (tid mod kTmChannels, tid / kTmChannels)
// copies element (time j + 32 k, channel c) for k = 0, 1, ... -- 64 contiguous bytes of a time row
// per 16 threads -- into / out of warp c's tile buffer.  No shift (nothing is wider than 4 bytes).
constexpr int kTmChannels = 16;
// distance between the shared-memory areas of two warps: = 4 (mod 32) floats in the time-major
// mapping, so that the 16 channels of one time sample fall into 8 different banks
template <int L, bool kTM> __host__ __device__ constexpr int warp_stride()
{
    return kTM ? warp_smem_floats<L>() + ((36 - warp_smem_floats<L>() % 32) % 32) : warp_smem_floats<L>();
}

// (addresses advance incrementally -- 32 time samples per step, a hop over the 16-byte pad whenever
// a lane region of 2L floats ends: these loops run once per element and must stay a few
// instructions long)
template <int L> struct TmWalk {
    static constexpr int R = 2 * L;                 // floats per lane region
    unsigned sa;                                    // shared-space byte address of the element
    int r;                                          // its position inside the lane region
    __device__ __forceinline__ TmWalk(int float_off, int e0)
    {
        sa = (unsigned)__cvta_generic_to_shared(&fk_smem[float_off + raw_index<L>(e0)]);
        r = e0 % R;
    }
    __device__ __forceinline__ void step()
    {
        sa += 128u + 16u * (32 / R);
        r += 32 % R;
        if (32 % R != 0 && r >= R) { r -= R; sa += 16u; }
    }
};

// The load of a tile is issued in portions (between the sections of the tile before it): 48
// four-byte copies per thread in one go fill the load/store queue and hold the warp up.
template <int L> struct TmPrefetch {
    TmWalk<L> w;
    const float* gp;
    const float* dummy;
    long long gstep;
    int t, n_t, left;
    bool chok, interior;
    __device__ __forceinline__ TmPrefetch(const PushParams<L>& p, const Chunk& ck, const Geom& g, int cg, int tile, int bufoff)
        : w((int)(threadIdx.x & (kTmChannels - 1)) * warp_stride<L, true>() + bufoff, (int)(threadIdx.x / kTmChannels))
    {
        const int c = threadIdx.x & (kTmChannels - 1), j = threadIdx.x / kTmChannels;
        const int ch = cg * kTmChannels + c;
        const int t0 = tile * Geo<L>::tile - g.r0;
        chok = ch < p.n_ch;
        gp = ck.in + ch + (long long)(t0 + j) * ck.in_pitch;
        dummy = ck.in;
        gstep = 32LL * ck.in_pitch;
        t = t0 + j; n_t = ck.n_t; left = Geo<L>::tile / 32;
        interior = chok && t0 >= 0 && t0 + Geo<L>::tile <= ck.n_t;
    }
    __device__ __forceinline__ void issue(int n)
    {
        n = min(n, left);
        left -= n;
        if (interior) {
#pragma unroll 2
            for (int k = 0; k < n; ++k) {
                asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(w.sa), "l"(gp) : "memory");
                gp += gstep; w.step();
            }
        } else {
#pragma unroll 2
            for (int k = 0; k < n; ++k) {
                const bool ok = chok && t < n_t;
                if (t >= 0)
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(w.sa), "l"(ok ? gp : dummy), "r"(ok ? 4 : 0) : "memory");
                gp += gstep; t += 32; w.step();
            }
        }
    }
    __device__ __forceinline__ void finish() { issue(left); cp_async_commit(); }
};

template <int L>
__device__ __forceinline__ void issue_tile_input_tm(const PushParams<L>& p, const Chunk& ck, const Geom& g, int cg, int tile, int bufoff)
{
    TmPrefetch<L> pf(p, ck, g, cg, tile, bufoff);
    pf.finish();
}

// Stores: thread (q, j) = (tid mod 4, tid / 4) gathers the samples of channels 4q .. 4q + 3 at time
// j + 128 k from four warps' buffers and writes them with one 16-byte store (8 time rows of 64 bytes
// per warp instruction) when the rows are 16-byte aligned (p.vec4), one by one otherwise.
template <int L>
__device__ __forceinline__ void store_tile_tm(const PushParams<L>& p, const Chunk& ck, const Geom& g, float* __restrict__ out, int cg,
                                              int bufoff, int t0)
{
    constexpr int S = warp_stride<L, true>();
    if (p.vec4 && (cg + 1) * kTmChannels <= p.n_ch) {
        const int q = threadIdx.x & 3, j = threadIdx.x >> 2;           // j = 0 .. 127
        const int t1 = min(ck.n_t - t0, Geo<L>::tile);                 // tile positions [max(0, -t0), t1) exist
        float* gp = out + (long long)cg * kTmChannels + 4 * q + (long long)(t0 + j) * ck.out_pitch;
        const long long gstep = 128LL * ck.out_pitch;
        const unsigned sa0 = (unsigned)__cvta_generic_to_shared(&fk_smem[4 * q * S + bufoff]);
#pragma unroll 2
        for (int e = j; e < Geo<L>::tile; e += 128) {
            if (e + t0 >= 0 && e < t1) {
                const unsigned sa = sa0 + 4u * (unsigned)raw_index<L>(e);
                float4 v;
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v.x) : "r"(sa));
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v.y) : "r"(sa + 4u * S));
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v.z) : "r"(sa + 8u * S));
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v.w) : "r"(sa + 12u * S));
                st_stream4(gp, v);
            }
            gp += gstep;
        }
        return;
    }
    const int c = threadIdx.x & (kTmChannels - 1), j = threadIdx.x / kTmChannels;
    const int ch = cg * kTmChannels + c;
    if (ch < p.n_ch) {
        TmWalk<L> w(c * S + bufoff, j);
        float* gp = out + ch + (long long)(t0 + j) * ck.out_pitch;
        const long long gstep = 32LL * ck.out_pitch;
        int t = t0 + j;
#pragma unroll 2
        for (int k = 0; k < Geo<L>::tile / 32; ++k) {
            if ((unsigned)t < (unsigned)ck.n_t) {
                float v;
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(w.sa));
                st_stream(gp, v);
            }
            gp += gstep; t += 32; w.step();
        }
    }
}

// S1: zero-state response of one section on the lane's two slots (the two halves of every
// pair); returns the end states s1 = (lo state 1, hi state 1), s2 = (lo state 2, hi state 2).
template <int L, int KIND>
__device__ __forceinline__ void local_pass(float2 (&x)[L], const SecParams<L>& T, float2& s1, float2& s2)
{
    const float c0 = T.c[0], c1 = T.c[1], c2 = T.c[2], c3 = T.c[3];
    s1 = s2 = make_float2(0.0f, 0.0f);
    if (KIND == kKindDF2) {
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const float2 w = fma2(c0, s1, fma2(c1, s2, x[i]));
            x[i] = fma2(c2, s1, fma2(c3, s2, w));
            s2 = s1; s1 = w;
        }
    } else if (KIND == kKindDelta || KIND == kKindDeltaG) {
        // u[n] = p u[n-1] - q w[n-1] + x[n] with w[n-1] = w[n-2] + u[n-1] substituted:
        // u[n] = (p - q) u[n-1] + (x[n] - q w[n-2]), so that one FMA per sample sits on the
        // critical path instead of three (c4 = p - q rounded from float64; 1 + a1 + a2 = q stays
        // exact).  wl lags one sample behind the state w.
        const float c4 = T.c[4];
        float2 wl = s2;
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const float2 t = fma2(c1, wl, x[i]);
            wl = add2(wl, s1);
            const float2 u = fma2(c4, s1, t);
            x[i] = fma2(c2, s1, u);
            if (KIND == kKindDeltaG) x[i] = fma2(c3, wl, x[i]);
            s1 = u;
        }
        s2 = add2(wl, s1);
    } else if (KIND == kKindNormal) {
        const float nc1 = -c1;
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const float2 xi = x[i];
            x[i] = fma2(c2, s1, fma2(c3, s2, xi));
            const float2 n1 = fma2(c0, s1, fma2(c1, s2, xi));
            s2 = fma2(c0, s2, mul2(f2(nc1), s1));
            s1 = n1;
        }
    } else {                                        // kKindDF2G: explicit b0 = coefficient 4
        const float c4 = T.c[4];
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const float2 w = fma2(c0, s1, fma2(c1, s2, x[i]));
            x[i] = fma2(c2, s1, fma2(c3, s2, mul2(f2(c4), w)));
            s2 = s1; s1 = w;
        }
    }
}

// Trigger on the characteristic function (reading R24 in DESIGN.md; PAPER.md:130
// "returns a list of time-channel-bounded events", :169 events may straddle chunks): per channel
//     off -> on  at the first sample with cf >= thr_on,   on -> off  at the first later one with cf < thr_off
// (an event (t_on, t_off, channel, peak cf) is appended to p.events when it closes), state carried with
// the channel's filter state.  Called for a tile only if it can matter (the channel is on, or some cf
// of the tile reaches thr_on): the cf of the tile lies in `buf` (lane regions, shift s), tile positions
// [e_lo, e_hi) are samples of this chunk, position e is sample g0 + e of the stream.  Every lane
// summarises its 2L samples; the warp then visits, in time order, only the lanes that can change the
// state (a lane with cf >= thr_on while off, one with cf < thr_off while on) and lets each walk its
// samples; the lanes passed over while on only raise the peak.
template <int L>
__device__ __noinline__ void trigger_tile(const PushParams<L>& p, int buf, int s, int wtr, int ch, long long g0,
                                          int e_lo, int e_hi, int lane)
{
    const float thr_on = p.thr_on, thr_off = p.thr_off;
    const int eb = 2 * L * lane;
    unsigned on = __float_as_uint(fk_smem[wtr]);
    float mx = 0.0f;
    bool has_on = false, has_off = false;
    for (int e = max(eb, e_lo); e < min(eb + 2 * L, e_hi); ++e) {
        const float c = fk_smem[buf + raw_index<L>(e + s)];
        mx = fmaxf(mx, c);
        has_on = has_on || c >= thr_on;
        has_off = has_off || c < thr_off;
    }
    const unsigned b_on = __ballot_sync(0xffffffffu, has_on), b_off = __ballot_sync(0xffffffffu, has_off);
    float peak = fk_smem[wtr + 1];
    long long t_on = (long long)(((unsigned long long)__float_as_uint(fk_smem[wtr + 3]) << 32) | __float_as_uint(fk_smem[wtr + 2]));
    const unsigned mxb = __float_as_uint(mx);               // (cf >= 0: the bit patterns order like the values)
    int last = -1;                                           // last lane that walked
    for (;;) {
        const unsigned cand = (on ? b_off : b_on) & (last >= 31 ? 0u : ~0u << (last + 1));
        const int l = cand ? __ffs((int)cand) - 1 : 32;
        if (on) {                                            // lanes passed over while on
            const bool mid = lane > last && lane < l;
            peak = fmaxf(peak, __uint_as_float(__reduce_max_sync(0xffffffffu, mid ? mxb : 0u)));
        }
        if (l == 32) break;
        if (lane == l) {
            for (int e = max(eb, e_lo); e < min(eb + 2 * L, e_hi); ++e) {
                const float c = fk_smem[buf + raw_index<L>(e + s)];
                if (!on) {
                    if (c >= thr_on) { on = 1u; t_on = g0 + e; peak = c; }
                } else if (c < thr_off) {
                    const unsigned idx = atomicAdd(p.n_events, 1u);
                    if (idx < p.ev_cap) p.events[idx] = Event{t_on, g0 + e, ch, peak};
                    on = 0u;
                } else {
                    peak = fmaxf(peak, c);
                }
            }
        }
        on = __shfl_sync(0xffffffffu, on, l);
        peak = __shfl_sync(0xffffffffu, peak, l);
        t_on = __shfl_sync(0xffffffffu, t_on, l);
        last = l;
    }
    if (lane == 0) {
        fk_smem[wtr] = __uint_as_float(on);
        fk_smem[wtr + 1] = peak;
        fk_smem[wtr + 2] = __uint_as_float((unsigned)((unsigned long long)t_on & 0xffffffffull));
        fk_smem[wtr + 3] = __uint_as_float((unsigned)((unsigned long long)t_on >> 32));
    }
    __syncwarp();
}

// One tile of one channel, samples already in x (gain applied): S1..S7.  `buf` stages the
// outputs.  buf / wst are float offsets into fk_smem.
// (kTM: time-major chunk; the CTA's warps hold the channels cg kTmChannels + warp and store together;
// `bufoff` = buf relative to the warp's shared-memory area; `item_end` is false for a warp whose
// channel does not exist)
// kForm: 0 = the two common section forms only, 1 = every section form, 2 / 3 = the same two + the trigger
// (filark_stream_set_trigger): a push kernel without a trigger set carries none of its code.
template <int L, bool kInterior, int kForm, bool kTM, bool kShift>
__device__ __forceinline__ void process_tile(const PushParams<L>& p, const Chunk& ck, const Geom& g, int buf, int wst, float2 (&x)[L],
                                             int ch, int tile, int lane, unsigned long long seen,
                                             bool item_end, unsigned rel_val, int cg, int bufoff,
                                             const TimeOrder<L>& to, TmPrefetch<L>* pf = nullptr)
{
    constexpr bool kAllKinds = (kForm & 1) != 0, kTrig = kForm >= 2;
    const bool last = tile == g.n_tiles - 1;
    const int t0 = tile * Geo<L>::tile - g.r0;
    // the carried state moves to the end of the tile's last FULL slot (slot q - 1)
    const int q = last ? g.q_last : 64;
    const bool keep = q == 0;
    const int jl = keep ? 0 : (q - 1) >> 1;
    const bool out_hi = ((q - 1) & 1) != 0;

    const unsigned wst_sa = smem_addr(wst);
    // (a running address for the carried state of the sections.  The section index k must not be needed in a
    // vector register: where it was -- as k-dependent shared-memory address -- ptxas kept the loop counter
    // in a vector register in some instantiations and then indexed every table per lane, with register
    // operands instead of uniform ones in all FFMA2 of the section loop: -30 %)
    unsigned sec_sa = wst_sa;
    // ---- S1..S3 per section -------------------------------------------------------------------
    const int pf_part = kTM ? (Geo<L>::tile / 32 + p.n_sec - 1) / p.n_sec : 0;
    for (int k = 0; k < p.n_sec; ++k) {
        const SecParams<L>& T = p.sec[k];
        float2 s1, s2;
        if (kTM && pf != nullptr) pf->issue(pf_part);
        // (kAllKinds = false: the kernel for cascades made of the two common section forms only --
        // what a Butterworth bandpass gives -- without the code of the other three)
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
        // S2: lane total W = P a + b (a, b: end states of the lo / hi slot from rest); the carried
        // state S enters lane 0's total through A^2L; inclusive scan over the lanes
        const float2 S = lds_f2(sec_sa);
        const float P0 = T.P[0], P1 = T.P[1], P2 = T.P[2], P3 = T.P[3];
        float W1 = fmaf(P0, s1.x, fmaf(P1, s2.x, s1.y)), W2 = fmaf(P2, s1.x, fmaf(P3, s2.x, s2.y));
        {
            // (selects instead of branches: the table operands stay uniform-register reads)
            const float S1 = lane == 0 ? S.x : 0.0f, S2 = lane == 0 ? S.y : 0.0f;
            W1 = fmaf(T.Q[0][0], S1, fmaf(T.Q[0][1], S2, W1));
            W2 = fmaf(T.Q[0][2], S1, fmaf(T.Q[0][3], S2, W2));
        }
        const int nsteps = T.nsteps;
        auto scan_step = [&](int d) {
            const float U1 = __shfl_up_sync(0xffffffffu, W1, 1 << d), U2 = __shfl_up_sync(0xffffffffu, W2, 1 << d);
            // (predicated updates instead of zeroed operands: two selects fewer per step)
            const float N1 = fmaf(T.Q[d][0], U1, fmaf(T.Q[d][1], U2, W1));
            const float N2 = fmaf(T.Q[d][2], U1, fmaf(T.Q[d][3], U2, W2));
            if (lane >= (1 << d)) { W1 = N1; W2 = N2; }
        };
        if (nsteps == kSteps) {                      // poles next to the unit circle: all steps, no tests
#pragma unroll
            for (int d = 0; d < kSteps; ++d) scan_step(d);
        } else {
#pragma unroll
            for (int d = 0; d < kSteps - 1; ++d)
                if (d < nsteps) scan_step(d);
        }
        float E1 = __shfl_up_sync(0xffffffffu, W1, 1), E2 = __shfl_up_sync(0xffffffffu, W2, 1);
        if (lane == 0) { E1 = S.x; E2 = S.y; }                      // state entering the lane's lo slot
        const float o1 = fmaf(P0, E1, fmaf(P1, E2, s1.x)), o2 = fmaf(P2, E1, fmaf(P3, E2, s2.x));   // ... its hi slot
        const float n1 = __shfl_sync(0xffffffffu, out_hi ? W1 : o1, jl);
        const float n2 = __shfl_sync(0xffffffffu, out_hi ? W2 : o2, jl);
        if (lane == 0 && !keep) sts_f2(sec_sa, make_float2(n1, n2));
        sec_sa += 8u;
        // S3 fix-up: y[i] += g1[i] s1 + g2[i] s2
        const float2 Ea = make_float2(E1, o1), Eb = make_float2(E2, o2);
        // (two rows per 16-byte uniform load: the tables are 16-byte aligned in the parameter bank)
#pragma unroll
        for (int i = 0; i < L; i += 2) {
            const float4 gg = *reinterpret_cast<const float4*>(&T.g[i][0]);
            x[i] = fma2(gg.x, Ea, fma2(gg.y, Eb, x[i]));
            x[i + 1] = fma2(gg.z, Ea, fma2(gg.w, Eb, x[i + 1]));
        }
    }

    if (kTM && pf != nullptr) pf->finish();
    if (ck.filt) {
        if (kTM) {
            regs_to_buf<L>(x, buf, lane, 0);
            __syncthreads();
            store_tile_tm<L>(p, ck, g, ck.filt, cg, bufoff, t0);
            __syncthreads();
        } else {
            float* row = ck.filt + (long long)ch * ck.out_pitch;
            const int sf = row_shift(row, g.r0);
            regs_to_buf<L>(x, buf, lane, sf);
            __syncwarp();
            store_tile<L, kInterior, kShift>(ck, g, row, buf, lane, t0, sf, to);
            __syncwarp();
        }
    }

    // ---- S4..S6: energy, the two averages, ratio --------------------------------------------
    const float as = p.avg.alpha[0], al = p.avg.alpha[1];
    float2 sp = make_float2(0.0f, 0.0f), lp = sp;                 // (lo slot, hi slot) from rest
#pragma unroll
    for (int i = 0; i < L; ++i) {
        const float2 e = mul2(x[i], x[i]);
        x[i] = e;
        sp = fma2(as, sp, e); lp = fma2(al, lp, e);
    }
    const int ks = wst + 2 * p.n_sec;
    const float2 M = lds_f2(sec_sa);                                           // carried (sta~, lta~)
    const float bLs = p.avg.betaL[0], bLl = p.avg.betaL[1];
    float Ws = sp.y + fmaf(-bLs, sp.x, sp.x), Wl = lp.y + fmaf(-bLl, lp.x, lp.x);        // alpha^L lo + hi
    {
        const float Ms = lane == 0 ? M.x : 0.0f, Ml = lane == 0 ? M.y : 0.0f;
        Ws += fmaf(-p.avg.betaQ[0][0], Ms, Ms); Wl += fmaf(-p.avg.betaQ[0][1], Ml, Ml);
    }
#pragma unroll
    for (int d = 0; d < kSteps; ++d) {
        const float Us = __shfl_up_sync(0xffffffffu, Ws, 1 << d), Ul = __shfl_up_sync(0xffffffffu, Wl, 1 << d);
        const float Ns_ = Ws + fmaf(-p.avg.betaQ[d][0], Us, Us), Nl_ = Wl + fmaf(-p.avg.betaQ[d][1], Ul, Ul);
        if (lane >= (1 << d)) { Ws = Ns_; Wl = Nl_; }
    }
    float Es = __shfl_up_sync(0xffffffffu, Ws, 1), El = __shfl_up_sync(0xffffffffu, Wl, 1);
    if (lane == 0) { Es = M.x; El = M.y; }
    const float Os = sp.x + fmaf(-bLs, Es, Es), Ol = lp.x + fmaf(-bLl, El, El);          // carry-in of the hi slot
    const float Ns = __shfl_sync(0xffffffffu, out_hi ? Ws : Os, jl);
    const float Nl = __shfl_sync(0xffffffffu, out_hi ? Wl : Ol, jl);
    if (lane == 0 && !keep) sts_f2(sec_sa, make_float2(Ns, Nl));

    // Last tile of a work item: the carried state is final here.  It goes back to global memory
    // now, and `progress` is released after the ratio loop below: the fence of the release waits for
    // the stores the warp has in flight, and by then these are a loop old (at the very end of the
    // tile, behind the cf stores, it cost about a microsecond per item).  What is stored after the
    // release are outputs only; nobody who waits on `progress` reads them (the host orders pushes
    // that share a buffer), the end of the grid publishes them.
    if (item_end) {
        __syncwarp();
        const int ns = state_floats(p.n_sec);
        float* gst = p.state + (long long)ch * ns;
        if (lane < ns) __stcg(gst + lane, fk_smem[wst + lane]);
        if (lane + 32 < ns) __stcg(gst + lane + 32, fk_smem[wst + lane + 32]);
    }

    if (ck.cf || kTrig) {
        // warm-up (reading R10): samples whose index since create/reset is < lta_len give cf = 0
        // (seen = samples pushed before this push; tile position e is sample seen + t0 + e of the stream)
        const long long rem = (long long)p.lta_len - (long long)seen - t0;     // first tile position with cf != 0
        const float ratio = p.ratio, thr = p.lta_thr;
        float2 Ps = make_float2(Es, Os), Pl = make_float2(El, Ol);
        // l~ never drops below alpha^L times its carry-in inside a slot (e >= 0)
        const bool live = fmaf(-bLl, El, El) > thr && fmaf(-bLl, Ol, Ol) > thr;
        if (rem <= 0 && __all_sync(0xffffffffu, live)) {
#pragma unroll
            for (int i = 0; i < L; ++i) {
                Ps = fma2(as, Ps, x[i]); Pl = fma2(al, Pl, x[i]);
                const float2 num = mul2(Ps, f2(ratio));
                x[i] = mul2(num, make_float2(rcp_fast(Pl.x), rcp_fast(Pl.y)));
            }
        } else {
            const int wm = rem > (1 << 30) ? (1 << 30) : (rem < 0 ? 0 : (int)rem);
            const int base = 2 * lane * L;
#pragma unroll
            for (int i = 0; i < L; ++i) {
                Ps = fma2(as, Ps, x[i]); Pl = fma2(al, Pl, x[i]);
                const float qa = (Ps.x * ratio) * rcp_fast(Pl.x), qb = (Ps.y * ratio) * rcp_fast(Pl.y);
                x[i].x = (Pl.x > thr && base + i >= wm) ? qa : 0.0f;
                x[i].y = (Pl.y > thr && base + L + i >= wm) ? qb : 0.0f;
            }
        }
        // trigger: does this tile matter?  Only if the channel is on, or some cf of the tile reaches thr_on
        // (positions outside the chunk included: that costs a needless visit at most)
        bool visit = false;
        if (kTrig) {
            float mx = fmaxf(x[0].x, x[0].y);
#pragma unroll
            for (int i = 1; i < L; ++i) mx = fmaxf(mx, fmaxf(x[i].x, x[i].y));
            visit = __any_sync(0xffffffffu, mx >= p.thr_on) || __float_as_uint(fk_smem[wst + trig_word(p.n_sec)]) != 0u;
        }
        const int sc = (kTM || !ck.cf) ? 0 : row_shift(ck.cf + (long long)ch * ck.out_pitch, g.r0);
        if (ck.cf || visit) {
            regs_to_buf<L>(x, buf, lane, sc);
            // (time-major: the CTA stores the cf together -- every warp is here; without a cf output only the warps
            // whose tile matters to the trigger are, each for its own buffer: a CTA barrier would never complete)
            if (kTM && ck.cf) __syncthreads(); else __syncwarp();
        }
        if (kTrig && visit && (!kTM || ch < p.n_ch)) {
            trigger_tile<L>(p, buf, sc, wst + trig_word(p.n_sec), ch, (long long)seen + t0, max(0, -t0),
                            min(Geo<L>::tile, ck.n_t - t0), lane);
            if (item_end && lane == 0) {             // (the state went back before the trigger ran)
                float* gtr = p.state + (long long)ch * state_floats(p.n_sec) + trig_word(p.n_sec);
                for (int j = 0; j < kTrigWords; ++j) __stcg(gtr + j, fk_smem[wst + trig_word(p.n_sec) + j]);
            }
        }
        if (item_end && lane == 0) st_release(p.progress + ch, rel_val);
        if (ck.cf) {
            if (kTM) store_tile_tm<L>(p, ck, g, ck.cf, cg, bufoff, t0);
            else store_tile<L, kInterior, kShift>(ck, g, ck.cf + (long long)ch * ck.out_pitch, buf, lane, t0, sc, to);
        }
    } else if (item_end) {
        __syncwarp();
        if (lane == 0) st_release(p.progress + ch, rel_val);
    }
    __syncwarp();
}


// Warps per SM (bounded by shared memory: two tile buffers per warp) and per CTA.  The kernel is
// built for two launch shapes: CTAS = kCmCtasPerSm small CTAs per SM for ordinary pushes, so that
// the CTAs of the next push can move in as soon as some of this push's CTAs have left, not only
// when the last warp of an SM is done; and CTAS = 1 (one CTA of all the SM's warps, warps of a CTA
// interleaved over the channels) for pushes long enough that the hand-over between pushes does
// not matter: with several CTAs per SM the hardware favours the older CTAs, the younger ones fall
// behind by 20 % and a long push ends with a tail (measured: 342 vs 377 Gsample/s on a 90,000-
// sample push).
constexpr int kCmCtasPerSm = 4;
#ifndef FK_MAXW16
#define FK_MAXW16 16
#endif
#ifndef FK_MAXW
#define FK_MAXW 16
#endif
template <int L> __host__ __device__ constexpr int cm_max_warps() { return L == 16 ? FK_MAXW16 : FK_MAXW; }
template <int L, int CTAS> __host__ __device__ constexpr int cm_cta_warps() { return cm_max_warps<L>() / CTAS; }

// Channel-major push: grid <= CTAS * SM count (every CTA of a push is resident once the
// pushes before it have drained), block = W * 32 (W <= cm_cta_warps<L, CTAS>()); dynamic shared memory =
// W * warp_smem_floats<L>() floats.
//
// Overlap of consecutive pushes.  A push of 6,000 channels x 1,500 samples is 2.5 tiles per
// resident warp and ~8 us of launch / first-load / drain latency that nothing inside one launch can
// hide.  The kernel is therefore launched with programmatic stream serialization and signals
// `launch_dependents` as soon as it has read its control slot: the CTAs of push e + 1 start on the
// SMs as the CTAs of push e leave, and the only ordering between the two is the real one -- channel
// c of push e + 1 starts from the state (and raw history) that push e left for channel c.
// `progress[c]` counts the segments completed on channel c since create/reset; item (seg, c) of a
// push whose slot says seq0 runs when progress[c] == seq0 + seg and then publishes seq0 + seg + 1
// (release at gpu scope, L2-scope polls).  At most kCmDepth pushes are in flight: push e starts only
// when push e - kCmDepth has completed (`exited`), so the host only has to compare a push's buffers
// with those of the kCmDepth - 1 pushes before it (p.wait_prior = 1 on a conflict, on another
// stream, after foreign work, or with FILARK_FLAG_STRICT_ORDER: then the kernel begins with
// griddepcontrol.wait like any dependent launch).  Every CTA ends with griddepcontrol.wait, so a push never completes before the
// push in front of it.
// kTM: time-major chunks through the transpose in shared memory (above): CTAS = 1, kTmChannels warps;
// the work items are (segment, group of kTmChannels channels) and belong to the CTA as a whole.
template <int L, int CTAS, int kForm, bool kTM, bool kDyn, bool kShift = false>
__global__ void __launch_bounds__(cm_cta_warps<L, CTAS>() * 32, CTAS)
filark_push_cm_kernel(const __grid_constant__ PushParams<L> p)
{
    // the warp index through a shuffle: the compiler then knows that it -- and with it the channel
    // walk, the section loop and every table index -- is warp-uniform, which is what lets the
    // tables be read through uniform registers
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31, W = blockDim.x >> 5;
    const int wbase = warp * warp_stride<L, kTM>();                   // two tile buffers, two state copies, history scratch
    const int wst0 = wbase + 2 * Geo<L>::buf_floats;
    const int whs = wst0 + 2 * kStateSmem;                            // history scratch
    const TimeOrder<L> to(lane);
    const int gw = kTM ? (int)(blockIdx.x * kTmChannels + warp)       // (time-major: the channel of the first item)
                       : CTAS == 1 ? (int)(blockIdx.x + gridDim.x * warp) : (int)(blockIdx.x * W + warp);   // warp index in the grid
    __shared__ unsigned sh_ctl[32];
    __shared__ unsigned sh_flag;
    __shared__ unsigned sh_item;
    __shared__ int sh_tile0[kMaxBatch + 1];          // tiles (per channel) of the launch in front of chunk k
    __shared__ unsigned sh_geo[kMaxBatch];           // slot geometry of chunk k: r0 | r1 << 8 | q_last << 16
    if (threadIdx.x == 0) sh_flag = 0u;

    if (p.wait_prior) asm volatile("griddepcontrol.wait;" ::: "memory");
    // the warp's first item is always (segment 0, channel gw): ask for its progress word now, so that
    // the answer is there when the control slot says what to compare it with
    // (static work distribution only: a claimed first item can be any channel)
    unsigned pr0 = 0;
    if (!kDyn && gw < p.n_ch) pr0 = ld_acquire(p.progress + gw);

    // ---- control slot of this push.  Nothing changes epoch or slot[epoch & 1] between the launch of
    // this grid (after every CTA of the previous push had taken its ticket and the last of them
    // had published both) and the last ticket of this grid: one 128-byte read by warp 0 suffices.
    CmCtl* const cc = p.cctl;
    if (warp == 0) {
        const unsigned* cw = reinterpret_cast<const unsigned*>(cc);
        unsigned v = ld_relaxed(cw + lane);
        const unsigned e = __shfl_sync(0xffffffffu, v, kCtlEpoch);
        const unsigned ring = __shfl_sync(0xffffffffu, v, kCtlSlotWords * (e & 1u) + 7);
        const unsigned need = __shfl_sync(0xffffffffu, v, kCtlSlotWords * (e & 1u) + 4 + ring);   // slot[e & 1].cum[ring]
        unsigned ex = __shfl_sync(0xffffffffu, v, kCtlExited + ring);
        // the chunks of this launch: chunk k starts r0_k = (r0 + samples in front of it) mod L samples
        // into a slot, which fixes its tiles (make_geom); an exclusive scan gives every chunk's first tile
        const unsigned R0 = __shfl_sync(0xffffffffu, v, kCtlSlotWords * (e & 1u) + 2);
        int carry = 0;
        for (int k0 = 0; k0 < p.n_push; k0 += 32) {
            const int k = k0 + lane;
            int inc = 0;
            unsigned geo = 0;
            if (k < p.n_push) {
                // (chunk 0 starts behind ALL samples waiting in the handle -- there can be more than L of
                // them after a launch with a longer L; every later chunk behind a partial slot)
                const unsigned r0k = k == 0 ? R0 : (R0 + p.ck[k].t_cum) % (unsigned)L;
                const Geom gk = make_geom<L>(r0k, p.ck[k].n_base, p.ck[k].n_rem, true);
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
        while ((int)(ex - need) < 0)                                   // push e - kCmDepth must have completed
            ex = __shfl_sync(0xffffffffu, ld_relaxed(&cc->exited[ring]), 0);
        sh_ctl[lane] = v;
    }
    __syncthreads();
    const unsigned epoch = sh_ctl[kCtlEpoch];
    const unsigned ring = sh_ctl[kCtlSlotWords * (epoch & 1u) + 7];
    const unsigned* sl = &sh_ctl[kCtlSlotWords * (epoch & 1u)];
    const unsigned long long seen = (unsigned long long)sl[0] | ((unsigned long long)sl[1] << 32);
    const unsigned seq0 = sl[3];
    const int ns = state_floats(p.n_sec);
    const int n_tiles_all = sh_tile0[p.n_push];          // tiles of the launch, per channel
    // chunk that holds tile gt of the launch (tiles are numbered through all chunks); warp-uniform
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

    // Work items (segment, channel), segment-major; a segment is seg_tiles consecutive tiles of a
    // channel (counted through all chunks of the launch), sized for about 8 items per warp.  Segment
    // s of a channel starts from the state its segment s - 1 left in global memory (`progress` says
    // when), i.e. item (s, c) waits for an item of LOWER index of the same launch (or, for s = 0,
    // for the launch before).
    //  - One segment per channel (ordinary pushes, kDyn = false): no waits inside the launch; warp gw takes
    //    items gw, gw + n_warps, ... statically.  What such a warp waits for belongs to an EARLIER launch,
    //    every CTA of which had started before this grid could launch.
    //  - Several segments per channel (long pushes and schedules, kDyn = true): items are CLAIMED from
    //    work[ring], a counter in the control block, in rising order.  The holder of a claimed item is
    //    therefore a resident warp, and so is the holder of every item it waits for (lower index =
    //    claimed earlier): the unfinished item of lowest index can always run, whether or not the other
    //    CTAs of the grid have been scheduled yet (two handles pushing on two streams share the SMs
    //    in any proportion).  The counter is never reset: launch e claims work[ring] - wbase[ring],
    //    and every warp (time-major: CTA) makes exactly two claims beyond the last item, so the
    //    next launch of this ring position starts at wbase + n_items + 2 claimers.
    const int n_warps = gridDim.x * W;
    const int seg_tiles = min(p.seg_tiles, n_tiles_all);
    const int n_seg = seg_tiles == n_tiles_all ? 1 : (n_tiles_all + seg_tiles - 1) / seg_tiles;
    const unsigned n_units = kTM ? (unsigned)((p.n_ch + kTmChannels - 1) / kTmChannels) : (unsigned)p.n_ch;
    const unsigned n_items = (unsigned)n_seg * n_units;
    constexpr bool dyn = kDyn;          // (chosen on the host: kDyn = false only if n_seg = 1 whatever r0 is)

    unsigned item = kTM ? blockIdx.x : (unsigned)gw;
    // Claimed items: the claim for the item AFTER the next one is always in flight (`pend`, raw counter
    // value, lane 0 of the warp / thread 0 of a time-major CTA), so that the round trip of the atomic
    // is never waited for except at the very start; every claimer ends with two claims beyond the
    // last item.  Holding an item while working on a lower one does not change the argument above.
    unsigned pend = 0;
    // (inline PTX on purpose: with the atomicAdd intrinsic here ptxas stops treating the loops around it
    // as warp-uniform in some instantiations and reads every table with per-lane loads, -30 %)
    auto claim_issue = [&]() {
        if (kTM ? threadIdx.x == 0 : lane == 0)
            asm volatile("atom.global.add.u32 %0, [%1], 1;" : "=r"(pend) : "l"(&cc->work[ring]) : "memory");
    };
    // (time-major: thread 0 publishes `pend` in sh_item before a CTA barrier, claim_take runs after it)
    // gt / gtend: first tile of the item and the tile behind its last, as tiles of the launch
    auto claim_take = [&](int& ch, int& gt, int& gtend, int& seg, int& cg) -> bool {
        unsigned it;
        if (dyn) {
            it = (kTM ? sh_item : __shfl_sync(0xffffffffu, pend, 0)) - sl[8 + ring];
        } else {
            it = item;
            item += kTM ? gridDim.x : (unsigned)n_warps;
        }
        if (it >= n_items) return false;
        seg = n_seg == 1 ? 0 : (int)(it / n_units);
        const int u = (int)(it - (unsigned)seg * n_units);
        cg = kTM ? u : 0;
        ch = kTM ? u * kTmChannels + warp : u;
        gt = seg * seg_tiles;
        gtend = min(n_tiles_all, gt + seg_tiles);
        return true;
    };
    // (every lane polls the same word and the value goes through a shuffle, so that the loop is
    // warp-uniform for the compiler: a divergent wait loop makes it give up the uniform-register
    // path for everything after it)
    auto wait_progress = [&](int ch, unsigned need, unsigned have_val) {
        unsigned done = __shfl_sync(0xffffffffu, have_val, 0);
        if ((int)(done - need) < 0) {
            do done = __shfl_sync(0xffffffffu, ld_relaxed(p.progress + ch), 0); while ((int)(done - need) < 0);
            (void)ld_acquire(p.progress + ch);       // (the acquire that goes with the release of the value the polls saw)
        }
    };

    int ch = 0, gt = 0, gtend = 0, seg = 0, cg = 0, cur = 0, wcur = 0, k = 0;
    // ---- hand the control block to the next launch, then let it start.  The ticket's round trip
    // runs while the first rows are requested; only warp 0 waits for it, the other warps look at
    // the flag when their first tile has arrived.
    unsigned tk = 0;
    if (warp == 0 && lane == 0) tk = atomicAdd(&cc->ticket, 1u);

    if (dyn) {
        claim_issue();
        if (kTM) { if (threadIdx.x == 0) sh_item = pend; __syncthreads(); }
    }
    bool have = claim_take(ch, gt, gtend, seg, cg);
    if (dyn) {
        if (kTM) __syncthreads();                    // (sh_item is rewritten at the next item's end)
        claim_issue();
    }
    if (have) {
        k = chunk_of(gt);
        const Geom g = geom_of(k);
        if (kTM) issue_tile_input_tm<L>(p, p.ck[k], g, cg, gt - sh_tile0[k], 0);
        else issue_tile_input<L, CTAS == 1, kShift>(p, p.ck[k], g, ch, gt - sh_tile0[k], wbase, lane, to);
        // the first segment of a channel needs what the previous launch left (state, hist): wait before
        // those loads are issued (a wait on an EARLIER launch cannot be part of a cycle)
        if (seg == 0 && ch < p.n_ch) {
            wait_progress(ch, seq0, kDyn ? ld_acquire(p.progress + ch) : pr0);
            issue_tile_carry<L>(p, g, ch, whs, wst0, lane);
        }
    }
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
                    __stcg(&nx->cum[j], sl[4 + j] + (j == ring ? gridDim.x : 0u));
                    __stcg(&nx->wbase[j], sl[8 + j] + (j == ring && dyn ? n_items + 2u * (kTM ? gridDim.x : (unsigned)n_warps) : 0u));
                }
                __stcg(&nx->ring, ring + 1u == (unsigned)kCmDepth ? 0u : ring + 1u);
                __stcg(&cc->ticket, 0u);
                st_release(&cc->epoch, epoch + 1u);
                __threadfence();
            }
            *reinterpret_cast<volatile unsigned*>(&sh_flag) = 1u;
        }
    }
    if (have) cp_async_wait_all();
    {
        unsigned f;
        do f = __shfl_sync(0xffffffffu, *reinterpret_cast<volatile unsigned*>(&sh_flag), 0); while (f == 0u);
    }
    asm volatile("griddepcontrol.launch_dependents;");

    while (have) {
        k = __shfl_sync(0xffffffffu, k, 0);            // (provably warp-uniform: the chunk is read through uniform registers)
        const Chunk& ck = p.ck[k];
        const Geom g = geom_of(k);
        const int tile = gt - sh_tile0[k];             // tile of the chunk
        int nch = ch, ngt = gt + 1, ngtend = gtend, nseg = seg, ncg = cg, nk = k;
        bool nhave = true;
        const bool item_end = ngt == gtend;
        const bool item_first = gt == seg * seg_tiles;
        const bool valid = !kTM || ch < p.n_ch;        // (time-major: the last group may have idle warps)
        unsigned npr = 0;
        if (item_end) {
            if (!dyn || !kTM) {
                nhave = claim_take(nch, ngt, ngtend, nseg, ncg);
                if (dyn) claim_issue();
                if (nhave && nseg == 0 && nch < p.n_ch) npr = ld_acquire(p.progress + nch);      // used after the tile is in registers
            } else if (threadIdx.x == 0) {
                sh_item = pend;
            }
        } else if (tile == g.n_tiles - 1) {
            nk = k + 1;                                // the item goes on in the next chunk
        }
        const int buf = wbase + cur * Geo<L>::buf_floats;
        const int wst = wst0 + wcur * kStateSmem;
        cp_async_wait_all();
        if (kTM) __syncthreads(); else __syncwarp();   // (time-major: every thread's part of the tile has landed)
        if (kTM && dyn && item_end) {
            nhave = claim_take(nch, ngt, ngtend, nseg, ncg);
            claim_issue();
            if (nhave && nseg == 0 && nch < p.n_ch) npr = ld_acquire(p.progress + nch);
        }
        if (item_end && nhave) nk = chunk_of(ngt);
        nk = __shfl_sync(0xffffffffu, nk, 0);
        if (valid && seg > 0 && item_first) {
            // first tile of a later segment: wait for the segment before it, then fetch its state (and,
            // where the segment begins with a chunk, the raw samples waiting in front of that chunk)
            wait_progress(ch, seq0 + (unsigned)seg, ld_acquire(p.progress + ch));
            const float* gst = p.state + (long long)ch * ns;
            if (lane < ns) fk_smem[wst + lane] = ld_relaxed_f32(gst + lane);
            if (lane + 32 < ns) fk_smem[wst + lane + 32] = ld_relaxed_f32(gst + lane + 32);
            if (tile == 0 && lane < g.r0) fk_smem[whs + lane] = ld_relaxed_f32(p.hist + (long long)ch * kHist + lane);
            __syncwarp();
        }
        const int sin = kTM ? 0 : row_shift(ck.in + (long long)ch * ck.in_pitch, g.r0);
        if (valid && tile == 0 && g.r0 != 0) {
            // first tile of the chunk: the waiting raw samples from the scratch to the head of the tile
            for (int e = lane; e < g.r0; e += 32) fk_smem[buf + raw_index<L>(e + sin)] = fk_smem[whs + e];
            __syncwarp();
        }
        if (valid && tile == g.n_tiles - 1 && g.r1 != 0) {
            // last tile of the chunk: keep the raw samples of its trailing partial slot -- in the scratch
            // if this item goes on with the next chunk, in the handle for whoever continues the channel
            const int e0 = g.q_last * L;                              // tile-space position of that slot
            if (item_end) {
                float* hd = p.hist + (long long)ch * kHist;
                for (int j = lane; j < g.r1; j += 32) hd[j] = fk_smem[buf + raw_index<L>(e0 + j + sin)];
            } else {
                for (int j = lane; j < g.r1; j += 32) fk_smem[whs + j] = fk_smem[buf + raw_index<L>(e0 + j + sin)];
            }
        }
        float2 x[L];
        buf_to_regs<L>(x, buf, lane, sin, p.gain);
        __syncwarp();
        if (nhave) {
            const int nbuf = wbase + (cur ^ 1) * Geo<L>::buf_floats;
            if (!kTM) issue_tile_input<L, CTAS == 1, kShift>(p, p.ck[nk], geom_of(nk), nch, ngt - sh_tile0[nk], nbuf, lane, to);
            if (item_end && nseg == 0 && nch < p.n_ch) {
                wait_progress(nch, seq0, npr);
                issue_tile_carry<L>(p, geom_of(nk), nch, whs, wst0 + (wcur ^ 1) * kStateSmem, lane);
            }
        }
        // (a segment's end writes the carried state back and tells whoever continues the channel:
        // the next segment of this launch or the first segment of the next launch)
        if (kTM) {
            // (time-major: the next tile is requested in portions while this one is computed)
            TmPrefetch<L> pf(p, p.ck[nk], geom_of(nk), ncg, ngt - sh_tile0[nk], (cur ^ 1) * Geo<L>::buf_floats);
            process_tile<L, true, kForm, true, false>(p, ck, g, buf, wst, x, ch, tile, lane, seen + ck.t_cum, item_end && valid,
                                                   seq0 + (unsigned)seg + 1u, cg, cur * Geo<L>::buf_floats, to,
                                                   nhave ? &pf : nullptr);
        } else {
            process_tile<L, CTAS == 1, kForm, false, kShift>(p, ck, g, buf, wst, x, ch, tile, lane, seen + ck.t_cum, item_end && valid,
                                                         seq0 + (unsigned)seg + 1u, cg, cur * Geo<L>::buf_floats, to);
        }
        if (item_end) wcur ^= 1;
        ch = nch; gt = ngt; gtend = ngtend; seg = nseg; cg = ncg; have = nhave; k = nk; cur ^= 1;
    }
    // completion: count this CTA out (push e + kCmDepth waits until all of them are)
    __syncthreads();
    if (threadIdx.x == 0)
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(&cc->exited[ring]) : "memory");
    // a push never completes before the push in front of it
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// Diagnostic kernel (FILARK_FLAG_SERIAL_SCAN, either layout): one thread per
// channel, serial in time, the same state-space sections, no blocked scan, no history: the
// carried state is the state after the last sample of the push.  Element (c, t) of a chunk is
// at c * sc + t * st; state word i of channel c is at c * state_sc + i * state_sk.
struct SerialParams {
    const float* in;
    float* filt;
    float* cf;
    float* state;
    long long n_t, sc_in, st_in, sc_out, st_out, state_sc, state_sk;
    int n_ch, n_sec, lta_len;
    float gain, ratio, lta_thr, inv_ns, inv_nl;
    int kind[kMaxSec];
    float c[kMaxSec][5];
};

__global__ void __launch_bounds__(128)
filark_push_serial_kernel(const __grid_constant__ SerialParams p)
{
    const int ch = blockIdx.x * blockDim.x + threadIdx.x;
    if (ch < p.n_ch) {
        float s[2 * kMaxSec + 2];
        const int nf = 2 * p.n_sec + 2;
        for (int i = 0; i < nf; ++i) s[i] = p.state[ch * p.state_sc + i * p.state_sk];
        const unsigned seen = __float_as_uint(p.state[ch * p.state_sc + nf * p.state_sk]);
        const float cs = p.inv_ns, cl = p.inv_nl;
        float ms = s[nf - 2], ml = s[nf - 1];
        for (long long t = 0; t < p.n_t; ++t) {
            float v = p.in[ch * p.sc_in + t * p.st_in] * p.gain;
            for (int k = 0; k < p.n_sec; ++k) {
                const int kind = p.kind[k];
                const float c0 = p.c[k][0], c1 = p.c[k][1], c2 = p.c[k][2], c3 = p.c[k][3], c4 = p.c[k][4];
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
            if (p.filt) p.filt[ch * p.sc_out + t * p.st_out] = v;
            const float e = v * v;
            ms = fmaf(-cs, ms, ms) + e;      // (1 - 1/N) m~ + e without rounding 1 - 1/N (reading R13)
            ml = fmaf(-cl, ml, ml) + e;
            if (p.cf)
                p.cf[ch * p.sc_out + t * p.st_out] =
                    (ml > p.lta_thr && (unsigned long long)seen + (unsigned long long)t >= (unsigned long long)p.lta_len)
                        ? p.ratio * __fdividef(ms, ml) : 0.0f;
        }
        s[nf - 2] = ms; s[nf - 1] = ml;
        for (int i = 0; i < nf; ++i) p.state[ch * p.state_sc + i * p.state_sk] = s[i];
        const unsigned long long s2 = (unsigned long long)seen + (unsigned long long)p.n_t;
        p.state[ch * p.state_sc + nf * p.state_sk] = __uint_as_float(s2 > kSeenMax ? kSeenMax : (unsigned)s2);
    }
}

}  // namespace filark
