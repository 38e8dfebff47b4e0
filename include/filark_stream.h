/*
 * filark_stream.h -- C ABI of the B200-native fused SOS + STA/LTA stream path.
 *
 * What the path computes (one "push" of a chunk of n_t samples on n_ch channels):
 *
 *   S0  load the chunk once from HBM (4 B/sample)
 *   S1  per SOS section, per time sub-block: zero-state local response      \
 *   S2  combine the sub-block transfer operators (warp-shuffle scan)         | stateful causal
 *   S3  fix-up with the carried state; new carried state kept in the handle /  SOS IIR filter
 *   S4  e = y^2
 *   S5  two exponential averages of e (STA, LTA) by the same local/scan/fix-up pattern
 *   S6  cf = sta/lta, 0 during the LTA warm-up and on dead channels
 *   S7  store filt and cf once (4 B + 4 B per sample)
 *
 * Source passages (PAPER.md = text of arxiv 2605.20132, "FiLark"):
 *   - PAPER.md:109 (sec. 3.4): IIR operators are "stateful-compatible", with "causal,
 *     sample-wise real-time variants (iir_filter_time_rt ...)" that "accept incremental
 *     data chunks and return outputs of matching length while maintaining correct state
 *     propagation internally".
 *   - PAPER.md:121 (Table 1): "IIR (offline & realtime second-order sections, SOS)".
 *   - PAPER.md:255 (sec. 6.2): state "is carried forward exactly"; only the first chunk
 *     after initialisation carries a transient.
 *   - PAPER.md:169 (sec. 3.5): state must propagate across file (= chunk) boundaries.
 *   - PAPER.md:83 (sec. 3.2): the filter leaves the underlying recording unchanged.
 *   - PAPER.md:130, 132 (sec. 3.4): the filtered stream feeds a streaming monitor such as a
 *     threshold-based energy detector.  The paper never defines STA/LTA; the characteristic
 *     function follows BASELINE.json `north_star` and the readings R8-R13 in DESIGN.md.
 *
 * Contract: concatenating the outputs of ANY sequence of pushes equals pushing the
 * concatenated input once (within the fp32 tolerance stated in DESIGN.md).
 *
 * All pointers named d_* are DEVICE pointers; everything else is a HOST pointer.
 * No exceptions cross this boundary, nothing aborts, nothing prints: every call returns a
 * filark_status_t.  A handle is bound to the CUDA device that was current at create and is
 * not thread-safe; pushes on one handle must be stream-ordered with respect to each other.
 */
#ifndef FILARK_STREAM_H
#define FILARK_STREAM_H

#ifdef __cplusplus
extern "C" {
#endif

/* Forward declaration so that this header needs no CUDA include. */
#ifndef __DRIVER_TYPES_H__
typedef struct CUstream_st *cudaStream_t;
#endif

typedef struct filark_stream filark_stream_t;   /* opaque; owns device state and tables */

typedef enum filark_status {
    FILARK_OK = 0,
    FILARK_ERR_INVALID_ARG = 1,     /* null pointer, non-positive size, bad layout/flags, aliasing */
    FILARK_ERR_UNSTABLE = 2,        /* a section has a pole with radius >= 1                       */
    FILARK_ERR_ALLOC = 3,           /* host or device allocation failed                            */
    FILARK_ERR_CUDA = 4,            /* a CUDA call failed; see filark_last_cuda_error              */
    FILARK_ERR_DEVICE_MISMATCH = 5, /* current device differs from the handle's device             */
    FILARK_ERR_ALIGNMENT = 6,       /* a device pointer is not 4-byte aligned                      */
    FILARK_ERR_TOO_LARGE = 7        /* filark_stream_once_noalloc: more channels than its fixed
                                       device scratch holds (FILARK_NOALLOC_MAX_CHANNELS)          */
} filark_status_t;

/* Memory order of a chunk (reading R14/R15 in DESIGN.md). */
#define FILARK_LAYOUT_CHANNEL_MAJOR 0   /* [n_ch][n_t]: time contiguous (BASELINE.json configs[0]) */
#define FILARK_LAYOUT_TIME_MAJOR    1   /* [n_t][n_ch]: channel contiguous (PAPER.md:160 'nt_nc')  */

/* create_ex flags */
#define FILARK_FLAG_NONE        0u
#define FILARK_FLAG_SERIAL_SCAN 1u  /* diagnostic kernel: one thread per channel, serial in time,
                                       same state-space arithmetic, no blocked scan             */

#define FILARK_FLAG_STRICT_ORDER 2u /* never overlap pushes, not even inside filark_stream_push_many
                                       (wins over FILARK_FLAG_OVERLAP_PUSHES)                     */

#define FILARK_FLAG_OVERLAP_PUSHES 4u /* the caller promises that, in the stream, NOTHING but this
                                       library's calls on this handle lies between one push and
                                       the next that writes the next push's input or touches its
                                       output buffers: consecutive push calls may then overlap on
                                       the device (see "Ordering" at filark_stream_push)         */

#define FILARK_FLAG_TM_TRANSPOSE 8u  /* tuning/testing, time-major chunks: always the kernel that transposes a
                                       tile through shared memory (one channel per warp), also where the
                                       kernel with one channel per lane would serve                    */

#define FILARK_FLAG_FORCE_L(L) ((unsigned)(L) << 8)  /* tuning/testing: use the kernel variant with
                                       sub-block length L (8, 16 or 24) for every push instead of
                                       the one chosen from n_t                                   */

#define FILARK_MAX_SECTIONS 16

/*
 * filark_stream_create -- build a stream for n_ch channels.
 *   out      [host, out]  receives the handle; untouched on error.
 *   n_ch     channels, >= 1.
 *   sos      [host, in]   row-major [n_sec][6] = b0 b1 b2 a0 a1 a2 per section, DOUBLE: fp32
 *                         coefficients alone break the tolerance for poles near z = 1
 *                         (DESIGN.md 4).  Sections are applied in the order given; each row is
 *                         divided by its a0.  Copied; the caller keeps ownership.
 *   n_sec    sections, 1 .. FILARK_MAX_SECTIONS.
 *   sta_len, lta_len  averaging lengths in SAMPLES, 1 <= sta_len <= lta_len (readings R8, R12).
 * Layout is channel-major, flags none.  Initial condition: zero state (reading R6).
 * Errors: INVALID_ARG (null, sizes, a0 == 0, non-finite coefficient), UNSTABLE, ALLOC, CUDA.
 * The handle owns n_ch*(2*n_sec+2) floats of device state plus a few KB of tables, allocated
 * on the current device.
 */
filark_status_t filark_stream_create(filark_stream_t **out, int n_ch, const double *sos, int n_sec,
                                     int sta_len, int lta_len);

/* Same, with the chunk layout (FILARK_LAYOUT_*) and flags (FILARK_FLAG_*). */
filark_status_t filark_stream_create_ex(filark_stream_t **out, int n_ch, const double *sos,
                                        int n_sec, int sta_len, int lta_len, int layout,
                                        unsigned flags);

/*
 * filark_stream_push -- filter one dense chunk and advance the carried state
 * ("accept incremental data chunks and return outputs of matching length";
 *  PAPER.md:255 state "carried forward exactly").
 *   d_in    [device, in]  n_ch*n_t floats in the handle's layout; never written.
 *   n_t     samples per channel in this chunk, >= 0; 0 is a no-op returning FILARK_OK.
 *   d_filt  [device, out] band-passed samples, same shape/layout as d_in; may be NULL.
 *   d_cf    [device, out] STA/LTA characteristic function, same shape/layout; may be NULL.
 *                         cf = 0 while fewer than lta_len samples have been seen since
 *                         create/reset, and where lta <= 1e-30 (readings R10, R11).
 *   stream  CUDA stream the work is enqueued on.
 * Asynchronous: enqueues exactly one kernel on `stream`, performs no host synchronisation and
 * no allocation, and may be captured into a CUDA graph.  The caller owns all three buffers and
 * keeps them alive until the stream reaches the push.  Outputs must not alias the input or
 * each other (in-place is rejected).
 * Ordering.  By default a push behaves like any kernel in `stream`: it sees all work enqueued
 * before it completed, and work enqueued after it sees the push (and all earlier pushes)
 * completed.  Consecutive pushes of one handle CAN overlap on the device -- the next push starts
 * while the previous one drains and orders itself against it channel by channel through the
 * carried state; at most three pushes of a handle are in flight and the outputs are bit-identical
 * either way -- but only where the library knows what lies between them in the stream:
 *   - between the pushes of one filark_stream_push_many call (nothing does), and
 *   - between separate push calls of a handle created with FILARK_FLAG_OVERLAP_PUSHES, by which
 *     the caller promises that no other work enqueued between two pushes produces the later
 *     push's input or touches its output buffers (the host cannot see foreign kernels, and a
 *     dependent launch that does not wait is not guaranteed to see their writes).
 * Even then a push waits like an ordinary kernel when the call before it in the stream (as far as
 * this library launched it) was not the same handle's push, or when it shares a buffer with the
 * two pushes before it (other than reading the same input).  Every push completes after all
 * earlier pushes of the handle.
 * Errors: INVALID_ARG (null handle/d_in, n_t < 0, both outputs NULL, aliasing), ALIGNMENT,
 * DEVICE_MISMATCH, CUDA (launch failure).
 */
filark_status_t filark_stream_push(filark_stream_t *h, const float *d_in, long long n_t,
                                   float *d_filt, float *d_cf, cudaStream_t stream);

/*
 * filark_stream_push_many -- enqueue a schedule of n_push consecutive dense chunks with one host
 * call (the pipeline executor's chunk loop; a folder of files is one
 * stream of chunks).  The same result as calling filark_stream_push n_push times in order (bit for
 * bit when the launches use the same sub-block length L, which is chosen per launch; to fp32
 * rounding otherwise, like any two chunkings of a record).  Chunks that share no buffer with each other are processed by COMMON launches of
 * up to 64 chunks (and < 2^31 samples per channel): every channel runs through all chunks of a
 * launch with its carried state held on the SM, so a chunk boundary inside a launch costs no
 * hand-over through device memory; consecutive launches of one call overlap on the device (see
 * "Ordering").  If an output of one chunk overlaps any buffer of another chunk, or with
 * FILARK_FLAG_STRICT_ORDER, every chunk gets a launch of its own, in order.
 *   d_in    [host, in]  n_push DEVICE pointers, chunk i holding n_ch*n_t[i] floats.
 *   n_t     [host, in]  n_push chunk lengths (>= 0; a zero-length chunk is skipped).
 *   d_filt, d_cf  [host, in]  n_push DEVICE pointers each; either array may be NULL (that output is
 *           not wanted for any chunk) and single entries may be NULL, but every chunk needs at
 *           least one output.
 * The whole schedule is checked before anything is enqueued: on an argument error nothing has been
 * launched.  Errors: as filark_stream_push.
 */
filark_status_t filark_stream_push_many(filark_stream_t *h, int n_push, const float *const *d_in,
                                        const long long *n_t, float *const *d_filt,
                                        float *const *d_cf, cudaStream_t stream);

/*
 * filark_stream_push_pitched -- as push, for a sub-view of a larger record: consecutive
 * rows of the chunk (rows = channels if channel-major, time samples if time-major) are
 * in_pitch / out_pitch ELEMENTS apart (>= the row length).  Both outputs share out_pitch.
 */
filark_status_t filark_stream_push_pitched(filark_stream_t *h, const float *d_in, long long n_t,
                                           long long in_pitch, float *d_filt, float *d_cf,
                                           long long out_pitch, cudaStream_t stream);

/*
 * filark_stream_push_host -- end-to-end variant for callers whose chunk lives in HOST memory
 * (the paper's pipeline executor hands the operator host arrays): copies the
 * dense chunk host->device into staging buffers owned by the handle, runs push on `stream`, and
 * copies the requested outputs device->host.  h_in / h_filt / h_cf are HOST pointers (pinned
 * memory for true asynchrony), n_ch*n_t floats each in the handle's layout; h_filt or h_cf may
 * be NULL.  The copies run on two streams owned by the handle (two alternating sets of staging
 * buffers), so that the upload of a chunk overlaps the download of the one before it; `stream`
 * is made to wait for the download, so the caller synchronises `stream` -- and nothing else --
 * before reading the outputs or changing h_in.  The staging buffers grow on demand: a push
 * larger than any before it synchronises and allocates (the only allocation in the push
 * family; not capturable in a CUDA graph).
 * Errors: as push, plus ALLOC.
 */
filark_status_t filark_stream_push_host(filark_stream_t *h, const float *h_in, long long n_t,
                                        float *h_filt, float *h_cf, cudaStream_t stream);

/*
 * filark_stream_reset -- return the handle to the just-created state (zero filter state, zero
 * sta/lta, sample counter 0), ordered on `stream` (the transient belongs to
 * "the first chunk processed after the filter is initialized").
 */
filark_status_t filark_stream_reset(filark_stream_t *h, cudaStream_t stream);

/*
 * Trigger / event emission on the characteristic function (the step behind S6: PAPER.md:130 a
 * monitor "consumes a data window and returns a list of time-channel-bounded events", :132
 * threshold-based detectors, :169 events may straddle chunk and file boundaries).  Classic on/off
 * trigger with hysteresis per channel (reading R24 in DESIGN.md), decided on the float32 cf:
 *     off -> on   at the first sample with cf >= thr_on
 *     on  -> off  at the first later sample with cf <  thr_off      (0 < thr_off <= thr_on)
 * An event is appended to a device list owned by the handle when it closes; the trigger state (on/off,
 * t_on, peak so far) is part of the carried state, so events straddle pushes.  The trigger runs inside
 * the push launches, behind the cf computation, also when d_cf is NULL (8 B/sample: input + filt, or
 * with d_filt = d_cf = NULL rejected as before -- one output array is still required).
 *
 * filark_stream_set_trigger -- thresholds and the capacity of the event list (>= 1 events; events
 *   closed while the list is full are dropped and counted).  thr_on = thr_off = 0 switches the
 *   trigger off.  Synchronises `stream` and the device; empties the list and sets every channel off.
 * filark_stream_pop_events  -- synchronises `stream`, copies the events closed so far to HOST memory
 *   (in no particular order: sort by (t_on, channel)) and empties the list.  *n_out = events copied,
 *   *n_dropped = events lost to a full list since the last pop (may be NULL).  If cap is smaller
 *   than the number of pending events nothing is consumed, *n_out says how many there are and the
 *   call returns INVALID_ARG.
 * Errors: INVALID_ARG, ALLOC, DEVICE_MISMATCH, CUDA.  filark_stream_reset and _set_state switch every
 * channel off but keep pending events.
 */
typedef struct filark_event {
    long long t_on;    /* index (samples since create/reset) of the first sample with cf >= thr_on */
    long long t_off;   /* index of the first later sample with cf < thr_off                         */
    int channel;
    float peak;        /* largest cf in [t_on, t_off)                                               */
} filark_event_t;
filark_status_t filark_stream_set_trigger(filark_stream_t *h, float thr_on, float thr_off,
                                          long long max_events, cudaStream_t stream);
filark_status_t filark_stream_pop_events(filark_stream_t *h, filark_event_t *out, long long cap,
                                         long long *n_out, long long *n_dropped, cudaStream_t stream);

/*
 * State export / import and the steady-state initial condition ("maintaining correct
 * state propagation"; :169 state survives file boundaries -- here: handles and processes;
 * :255 "a short transient determined by the filter order and the initial condition").
 *
 * filark_stream_state_size -- bytes of this handle's state blob: 64 + n_ch * (2 n_sec + 2) * 8.
 * filark_stream_get_state  -- synchronises `stream` (and the device), writes the blob to HOST memory.
 *   Layout: 64-byte header {"FKSTATE1", int n_ch, n_sec, sta_len, lta_len, uint64 samples seen,
 *   32 reserved bytes}, then per channel 2 n_sec + 2 doubles: the state s_k of every section k in
 *   the coordinates filark_debug_design reports (s[n] = A s[n-1] + B x[n], y[n] = C s[n-1] + D x[n],
 *   the cascade's gain in front of section 0) after the LAST pushed sample, then sta * sta_len and
 *   lta * lta_len.  (Inside the handle the state stands at a sub-block boundary with up to 23 raw
 *   samples waiting; the export runs those over it in float64, so the blob has no pending samples.)
 * filark_stream_set_state  -- the reverse, into a handle created with the same n_ch, n_sec, sta_len,
 *   lta_len (and, for the outputs to continue, the same sos): pushing B after importing the state
 *   exported behind A gives the outputs of A || B to fp32 rounding.  Synchronises.
 * filark_stream_set_initial_condition -- the state every channel would have if its input had been
 *   the constant x0[c] (HOST array, n_ch floats) for ever: s = (I - A)^-1 B v per section, the
 *   averages at the steady energy, the warm-up over (scipy's `zi = sosfilt_zi(sos) * x0` idiom).
 *   create/reset give the zero state (reading R6).  Synchronises.
 * Errors: INVALID_ARG (null, blob too small or of another handle shape, non-finite values, handle
 * with FILARK_FLAG_SERIAL_SCAN), DEVICE_MISMATCH, CUDA.
 */
long long filark_stream_state_size(const filark_stream_t *h);
filark_status_t filark_stream_get_state(filark_stream_t *h, void *blob, long long size, cudaStream_t stream);
filark_status_t filark_stream_set_state(filark_stream_t *h, const void *blob, long long size, cudaStream_t stream);
filark_status_t filark_stream_set_initial_condition(filark_stream_t *h, const float *x0, cudaStream_t stream);

/*
 * filark_events_associate -- per-channel events -> time-channel-bounded events ("a list of
 * time-channel-bounded events", :132 "each described by a time and channel extent"; SURVEY.md 8(f) NEXT-1
 * "(t_on, t_off, channel range, peak cf)").  The paper gives no rule; reading R30 in DESIGN.md:
 *   two events are linked if their channels differ by at most ch_gap and their half-open intervals
 *   [t_on, t_off) come within t_gap samples of each other (t_on1 < t_off2 + t_gap and t_on2 < t_off1 +
 *   t_gap; t_gap = 0: they overlap); a box is a connected component of the link graph: the smallest t_on,
 *   the largest t_off, the channel extent [ch_lo, ch_hi], the largest peak, the number of events.
 * HOST function on a HOST list (what filark_stream_pop_events returned, in any order; the list is compact --
 * about 10^4 events per minute of a 6,000-channel fibre): a sweep in rising t_on over per-channel lists of
 * the events still within reach, union-find for the components.  `boxes` receives at most `cap` boxes in
 * rising (t_on, ch_lo, t_off, ch_hi); *n_boxes the number found (larger than cap: the rest is dropped).
 * Touches no device.  Errors: INVALID_ARG (null, negative count or gap), ALLOC (host memory).
 */
typedef struct filark_box {
    long long t_on, t_off;   /* [t_on, t_off): sample indices since create/reset */
    int ch_lo, ch_hi;        /* channel extent, inclusive */
    float peak;              /* largest cf of its events */
    int n_events;
} filark_box_t;
filark_status_t filark_events_associate(const filark_event_t *events, long long n, int ch_gap, long long t_gap,
                                        filark_box_t *boxes, long long cap, long long *n_boxes);

/*
 * filark_stream_zero_phase -- the zero-phase mode of the display filter ("Implemented as
 * either a zero-phase or causal IIR filter ... applied only to the currently visible buffer"): the
 * handle's cascade run forward over a bounded window, the result reversed in time, run again, and
 * reversed back; each pass starts from the steady state of the first sample of its input, there is no
 * padding (reading R29: scipy's sosfiltfilt(..., padtype=None)).  d_in, d_out: dense windows of n_ch x
 * n_t floats in the handle's layout (d_out may equal d_in).  Does NOT touch the carried state of the
 * stream (a second stream of the same cascade and two window-sized temporaries are made on first use
 * and grow on demand: the only allocations; a larger window synchronises).  Enqueues six kernels on
 * `stream`.  Errors: INVALID_ARG, ALIGNMENT, ALLOC, DEVICE_MISMATCH, CUDA.
 */
filark_status_t filark_stream_zero_phase(filark_stream_t *h, const float *d_in, long long n_t, float *d_out,
                                         cudaStream_t stream);

/*
 * filark_stream_once_noalloc -- the whole path S0..S7 over ONE dense record from rest, without a handle and
 * WITHOUT ANY ALLOCATION: for callers that cannot call cudaMalloc (a CUDA graph being captured, a tight
 * serving loop, a harness that forbids it).  The result is what filark_stream_create_ex + one
 * filark_stream_push of the same record give (the same kernel runs), e.g. the characteristic function of
 * a window of channels x samples.
 *
 * What a handle keeps in device memory of its own -- the carried state, the raw-history rows, the
 * per-channel progress words and the control block of the push kernel -- lives here in ONE fixed array in
 * the library's device image (`static __device__`, FILARK_NOALLOC_SCRATCH_BYTES = 6.6 MiB, held by every
 * GPU that loads the library until the process exits), sized for FILARK_NOALLOC_MAX_CHANNELS channels.
 * More channels are refused with FILARK_ERR_TOO_LARGE (shard the channels over several calls, or use a
 * handle).  The call enqueues, on `stream`: three memsets that put the part of the array it uses back to
 * zero (the array keeps what the previous call left), then one launch of the push kernel.  The cascade is
 * designed on the host in the call (float64, about 0.1 ms for eight sections); no cudaMalloc, cudaFree or
 * other allocating CUDA routine is called, nothing is synchronised.
 *
 * EVERY call on a device shares that array.  Calls in one stream follow one another and are safe; calls
 * that can overlap on the GPU (different streams without an ordering between them, several host threads)
 * RACE on it and give wrong results: order them yourself.  Handles do not use the array.
 *
 *   sos, n_sec, sta_len, lta_len, layout   as filark_stream_create_ex (flags: none)
 *   d_in    n_ch x n_t floats, dense, in `layout`; d_filt / d_cf: the same shape, either may be NULL (not
 *           both); none may overlap another.  n_t >= 0 (0: no-op).
 *   cuda_error   may be NULL; receives the cudaError_t (as int) of a failing CUDA call.
 * Errors: INVALID_ARG, UNSTABLE, ALIGNMENT, TOO_LARGE, CUDA.
 */
#define FILARK_NOALLOC_MAX_CHANNELS 16384
#define FILARK_NOALLOC_SCRATCH_BYTES (FILARK_NOALLOC_MAX_CHANNELS * 420 + 256)
filark_status_t filark_stream_once_noalloc(const double *sos, int n_sec, int sta_len, int lta_len, int layout,
                                           const float *d_in, int n_ch, long long n_t, float *d_filt,
                                           float *d_cf, cudaStream_t stream, int *cuda_error);

/* Free the handle and its device memory (on the handle's device, whichever device is current).
 * NULL is accepted.  Synchronises the handle's device. */
filark_status_t filark_stream_destroy(filark_stream_t *h);

/* Static description of a status code; never NULL. */
const char *filark_status_string(filark_status_t s);

/* The cudaError_t (as int) of the last failing CUDA call on this handle, 0 if none. */
int filark_last_cuda_error(const filark_stream_t *h);

/*
 * Introspection used by the harness: number of kernels launched so far through this handle
 * (bench.py reports it as gpu_launches) and the number of samples per channel pushed since
 * create/reset as tracked on the host.
 */
long long filark_stream_launch_count(const filark_stream_t *h);
long long filark_stream_samples_pushed(const filark_stream_t *h);

#ifdef __cplusplus
}
#endif
#endif /* FILARK_STREAM_H */
