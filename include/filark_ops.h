/*
 * filark_ops.h -- C ABI of the two small operators that sit beside the fused SOS + STA/LTA stream
 * path (include/filark_stream.h) and share its conventions: device pointers are named d_*, every
 * call returns a filark_status_t, nothing aborts or prints, work is enqueued on the caller's stream.
 *
 * NEXT-3: streaming first-order operators through the same blocked 1-D scan as the
 *   STA/LTA averages -- PAPER.md:121 (Table 1) "running automatic gain control (AGC), running mean
 *   ... (all with stateful streaming variants)", :122 "gain equalisation (streaming exponential
 *   moving average, EMA variant)".  The paper gives no formula; reading R26 in DESIGN.md: with the
 *   exponential average m[n] = m[n-1] + (u[n] - m[n-1]) / N, state carried across pushes, zero at
 *   create/reset,
 *       FILARK_EMA_MEAN    u = x,    out = m            (running mean)
 *       FILARK_EMA_DEMEAN  u = x,    out = x - m        (running mean removed)
 *       FILARK_EMA_AGC     u = |x|,  out = x / (m + eps)
 *   Pushing a record in any chunking gives the same output as pushing it whole (fp32 rounding).
 *
 * NEXT-4: display decimation -- PAPER.md:171 (sec. 3.5) "logical downsampling is applied to match
 *   the display resolution ... drop mode preserves transient peaks, peak mode maintains amplitude
 *   envelopes, and linear interpolation smooths slowly varying wavefields".  Reading R25: `width`
 *   display columns per channel, column j covering input samples [a_j, a_{j+1}), a_j =
 *   floor(j n_t / width) (at least sample a_j),
 *       FILARK_DECIMATE_DROP    out[j] = x[a_j]
 *       FILARK_DECIMATE_PEAK    out[j] = the sample of largest magnitude of the column (the first one
 *                               on ties), with its sign
 *       FILARK_DECIMATE_LINEAR  out[j] = x at position j (n_t - 1) / (width - 1), linearly interpolated
 *   into a plain device buffer (no graphics API is involved anywhere in this repository).
 */
#ifndef FILARK_OPS_H
#define FILARK_OPS_H

#include "filark_stream.h"

#ifdef __cplusplus
extern "C" {
#endif

#define FILARK_EMA_MEAN   0
#define FILARK_EMA_DEMEAN 1
#define FILARK_EMA_AGC    2

typedef struct filark_ema filark_ema_t;   /* opaque; owns one float of device state per channel */

/*
 * filark_ema_create -- n_ch channels, averaging length n_len >= 1 samples, mode FILARK_EMA_*,
 * eps >= 0 (AGC only), layout FILARK_LAYOUT_* of the chunks.  State zero.  Bound to the current device.
 * Errors: INVALID_ARG, ALLOC, CUDA.
 */
filark_status_t filark_ema_create(filark_ema_t **out, int n_ch, int n_len, int mode, float eps, int layout);

/*
 * filark_ema_push -- one dense chunk of n_t >= 0 samples per channel ([n_ch][n_t] or [n_t][n_ch]):
 * d_out (same shape; may equal d_in: every sample is read before it is written) and the carried state.
 * One kernel on `stream`, no host synchronisation.  Errors: INVALID_ARG, ALIGNMENT, DEVICE_MISMATCH, CUDA.
 */
filark_status_t filark_ema_push(filark_ema_t *h, const float *d_in, long long n_t, float *d_out, cudaStream_t stream);

/* Zero state, ordered on `stream`. */
filark_status_t filark_ema_reset(filark_ema_t *h, cudaStream_t stream);
filark_status_t filark_ema_destroy(filark_ema_t *h);

#define FILARK_DECIMATE_DROP   0
#define FILARK_DECIMATE_PEAK   1
#define FILARK_DECIMATE_LINEAR 2

/*
 * filark_decimate -- stateless.  d_in: n_ch channels x n_t samples, rows `pitch` elements apart
 * (channel-major: element (c, n) at c*pitch + n, pitch >= n_t; time-major: at n*pitch + c, pitch >=
 * n_ch).  d_out: dense, [n_ch][width] (channel-major) or [width][n_ch] (time-major); must not overlap
 * d_in.  One kernel on `stream`.  Errors: INVALID_ARG (null, sizes < 1, unknown mode or layout,
 * overlap), ALIGNMENT (pointers not 4-byte aligned), CUDA.
 */
filark_status_t filark_decimate(const float *d_in, int n_ch, long long n_t, long long pitch, int layout,
                                int mode, int width, float *d_out, cudaStream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* FILARK_OPS_H */
