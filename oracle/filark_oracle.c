/*
 * filark_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, float64 CPU oracle for the one hot path this repository builds:
 * stateful chunked temporal filtering of a channel x time DAS stream =
 * per-channel cascaded second-order-section (SOS) IIR filter with state carried
 * across chunk boundaries, followed by a recursive STA/LTA characteristic
 * function (CF) with its own carried state.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or constant with paper_2605_20132_b200/csrc (the CUDA path).
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md):
 *  - PAPER.md:109 (section 3.4): IIR operators are "stateful-compatible",
 *    "causal, sample-wise real-time variants" that "accept incremental data
 *    chunks and return outputs of matching length while maintaining correct
 *    state propagation internally".
 *  - PAPER.md:121 (Table 1): "IIR (offline & realtime second-order sections, SOS)".
 *  - PAPER.md:255 (section 6.2): state "is carried forward exactly"; the first
 *    chunk after initialisation carries a transient "determined by the filter
 *    order and the initial condition" -> reading R6: zero initial state.
 *  - PAPER.md:130 (section 3.4): monitors such as a "threshold-based energy
 *    detector" consume the stream; the paper never defines STA/LTA, so the CF
 *    follows BASELINE.json north_star ("recursive STA/LTA characteristic
 *    function (also with carried state)") with readings R8-R13 of SURVEY.md 8(c).
 *
 * The method reaches exactly (up to rounding order) a result with a plain
 * definition -- a causal LTI cascade and two exponential averages -- so the
 * oracle is that definition written out, sample by sample, in double:
 *
 *   for each channel c (independent), state zero at create/reset:
 *     for each sample n (g = samples since create/reset, counted across pushes):
 *       v = (double) x[c][n]
 *       for k = 0 .. n_sec-1 (given order; b*,a* divided by a0_k once):   (R1,R4,R5)
 *           y     = b0_k*v + z1[k]               transposed direct form II
 *           z1[k] = b1_k*v - a1_k*y + z2[k]
 *           z2[k] = b2_k*v - a2_k*y
 *           v = y
 *       filt[c][n] = (float) v                   round to nearest           (R18)
 *       e   = v*v                                unrounded double v         (R9)
 *       sta = sta + (e - sta)/sta_len            both use current sample    (R8,R13)
 *       lta = lta + (e - lta)/lta_len
 *       cf[c][n] = (g >= lta_len && lta > 1e-30) ? (float)(sta/lta) : 0     (R10,R11)
 *
 * No blocking, fusion or reordering.  Compile WITHOUT -ffast-math and with
 * -ffp-contract=off so that every operation is an IEEE double operation in the
 * order written (chunked == whole must be bit-identical).
 *
 * Pins (tests/test_oracle_pins.py): closed-form biquad impulse response, zero
 * gain at DC and Nyquist, |H|^2 = 1/2 at the band edges, linearity,
 * bit-identical chunk invariance, brute-force expanded difference equation,
 * scipy.signal.sosfilt / lfilter special cases, STA/LTA closed forms, CF bound
 * and scale invariance.  The composition SOS -> y^2 -> STA/LTA -> ratio has no
 * closed form of its own: it is pinned through its parts.
 */
#include <stdlib.h>
#include <string.h>

#define FILARK_ORACLE_LTA_TINY 1e-30

typedef struct filark_oracle {
    int n_ch;
    int n_sec;
    int sta_len;
    int lta_len;
    double *coef;   /* [n_sec][5] = b0 b1 b2 a1 a2, already divided by a0 */
    double *z;      /* [n_ch][n_sec][2]  DF2T state z1, z2                */
    double *sta;    /* [n_ch]                                            */
    double *lta;    /* [n_ch]                                            */
    long long g;    /* samples pushed since create/reset                 */
} filark_oracle_t;

/* sos: row-major [n_sec][6] = b0 b1 b2 a0 a1 a2 (scipy convention). */
filark_oracle_t *filark_oracle_create(int n_ch, const double *sos, int n_sec,
                                      int sta_len, int lta_len)
{
    if (n_ch <= 0 || n_sec <= 0 || !sos || sta_len < 1 || lta_len < sta_len) return NULL;
    for (int k = 0; k < n_sec; ++k)
        if (sos[6 * k + 3] == 0.0) return NULL;
    filark_oracle_t *o = (filark_oracle_t *)calloc(1, sizeof(*o));
    if (!o) return NULL;
    o->n_ch = n_ch; o->n_sec = n_sec; o->sta_len = sta_len; o->lta_len = lta_len;
    o->coef = (double *)malloc(sizeof(double) * 5 * (size_t)n_sec);
    o->z    = (double *)calloc((size_t)n_ch * (size_t)n_sec * 2, sizeof(double));
    o->sta  = (double *)calloc((size_t)n_ch, sizeof(double));
    o->lta  = (double *)calloc((size_t)n_ch, sizeof(double));
    if (!o->coef || !o->z || !o->sta || !o->lta) {
        free(o->coef); free(o->z); free(o->sta); free(o->lta); free(o);
        return NULL;
    }
    for (int k = 0; k < n_sec; ++k) {
        const double a0 = sos[6 * k + 3];
        o->coef[5 * k + 0] = sos[6 * k + 0] / a0;
        o->coef[5 * k + 1] = sos[6 * k + 1] / a0;
        o->coef[5 * k + 2] = sos[6 * k + 2] / a0;
        o->coef[5 * k + 3] = sos[6 * k + 4] / a0;
        o->coef[5 * k + 4] = sos[6 * k + 5] / a0;
    }
    o->g = 0;
    return o;
}

void filark_oracle_reset(filark_oracle_t *o)
{
    if (!o) return;
    memset(o->z, 0, sizeof(double) * (size_t)o->n_ch * (size_t)o->n_sec * 2);
    memset(o->sta, 0, sizeof(double) * (size_t)o->n_ch);
    memset(o->lta, 0, sizeof(double) * (size_t)o->n_ch);
    o->g = 0;
}

void filark_oracle_destroy(filark_oracle_t *o)
{
    if (!o) return;
    free(o->coef); free(o->z); free(o->sta); free(o->lta); free(o);
}

long long filark_oracle_samples_seen(const filark_oracle_t *o) { return o ? o->g : -1; }

/*
 * Process channels [ch_begin, ch_end) of one chunk of n_t samples WITHOUT
 * advancing the sample counter (so that a caller may split the channel range
 * over threads; channels are independent).  Element (c, n) of x / filt / cf
 * lives at index c*stride_c + n*stride_n (in elements): channel-major dense
 * chunk = (n_t, 1), time-major dense chunk = (1, n_ch).  filt or cf may be NULL.
 */
int filark_oracle_push_range(filark_oracle_t *o, const float *x, long long n_t,
                             long long stride_c, long long stride_n,
                             float *filt, float *cf, int ch_begin, int ch_end)
{
    if (!o || !x || n_t < 0 || ch_begin < 0 || ch_end > o->n_ch || ch_begin > ch_end) return 1;
    const int n_sec = o->n_sec;
    const double sta_len = (double)o->sta_len;
    const double lta_len = (double)o->lta_len;
    for (int c = ch_begin; c < ch_end; ++c) {
        double *z = o->z + (size_t)c * (size_t)n_sec * 2;
        double sta = o->sta[c];
        double lta = o->lta[c];
        long long g = o->g;
        for (long long n = 0; n < n_t; ++n) {
            const long long idx = (long long)c * stride_c + n * stride_n;
            double v = (double)x[idx];
            for (int k = 0; k < n_sec; ++k) {
                const double *q = o->coef + 5 * k;     /* b0 b1 b2 a1 a2 */
                const double y = q[0] * v + z[2 * k];
                z[2 * k]     = q[1] * v - q[3] * y + z[2 * k + 1];
                z[2 * k + 1] = q[2] * v - q[4] * y;
                v = y;
            }
            if (filt) filt[idx] = (float)v;
            const double e = v * v;
            sta = sta + (e - sta) / sta_len;
            lta = lta + (e - lta) / lta_len;
            if (cf)
                cf[idx] = (g >= (long long)o->lta_len && lta > FILARK_ORACLE_LTA_TINY)
                              ? (float)(sta / lta) : 0.0f;
            g += 1;
        }
        o->sta[c] = sta;
        o->lta[c] = lta;
    }
    return 0;
}

/* Advance the sample counter once every channel range of the chunk is done. */
void filark_oracle_advance(filark_oracle_t *o, long long n_t)
{
    if (o && n_t > 0) o->g += n_t;
}

/* One whole push: all channels, then advance the counter. */
int filark_oracle_push(filark_oracle_t *o, const float *x, long long n_t,
                       long long stride_c, long long stride_n, float *filt, float *cf)
{
    if (!o) return 1;
    const int rc = filark_oracle_push_range(o, x, n_t, stride_c, stride_n, filt, cf, 0, o->n_ch);
    if (rc == 0) filark_oracle_advance(o, n_t);
    return rc;
}

/* Expose the float64 intermediates for pins that need them unrounded:
 * runs ONE channel of double input through the cascade + averages and returns
 * y (double), sta, lta per sample.  Same statements as above. */
int filark_oracle_trace_f64(filark_oracle_t *o, int c, const double *x, long long n_t,
                            double *y_out, double *sta_out, double *lta_out)
{
    if (!o || !x || c < 0 || c >= o->n_ch || n_t < 0) return 1;
    const int n_sec = o->n_sec;
    double *z = o->z + (size_t)c * (size_t)n_sec * 2;
    double sta = o->sta[c], lta = o->lta[c];
    for (long long n = 0; n < n_t; ++n) {
        double v = x[n];
        for (int k = 0; k < n_sec; ++k) {
            const double *q = o->coef + 5 * k;
            const double y = q[0] * v + z[2 * k];
            z[2 * k]     = q[1] * v - q[3] * y + z[2 * k + 1];
            z[2 * k + 1] = q[2] * v - q[4] * y;
            v = y;
        }
        const double e = v * v;
        sta = sta + (e - sta) / (double)o->sta_len;
        lta = lta + (e - lta) / (double)o->lta_len;
        if (y_out) y_out[n] = v;
        if (sta_out) sta_out[n] = sta;
        if (lta_out) lta_out[n] = lta;
    }
    o->sta[c] = sta; o->lta[c] = lta;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Additions for the NEXT rows of SURVEY.md 8(f) (nothing above this line was changed).
 * ------------------------------------------------------------------------------------------ */

/*
 * Steady-state initial condition ("a short transient determined
 * by the filter order and the initial condition"): the state every channel would have if its
 * input had been the constant x0[c] for ever.  For one transposed-direct-form-II section with
 * constant input v the output is y = v (b0+b1+b2)/(1+a1+a2) and the state follows from the two
 * update statements of the push loop read as fixed-point equations:
 *     z2 = b2 v - a2 y,      z1 = b1 v - a1 y + z2.
 * The averages start at the steady energy y_last^2, and the warm-up counter at lta_len (the
 * averages ARE warmed up).  This is scipy's `sosfilt_zi(sos) * x0` idiom, which pins it.
 */
int filark_oracle_set_initial_condition(filark_oracle_t *o, const double *x0)
{
    if (!o || !x0) return 1;
    for (int c = 0; c < o->n_ch; ++c) {
        double v = x0[c];
        double *z = o->z + (size_t)c * (size_t)o->n_sec * 2;
        for (int k = 0; k < o->n_sec; ++k) {
            const double *q = o->coef + 5 * k;     /* b0 b1 b2 a1 a2 */
            const double y = v * (q[0] + q[1] + q[2]) / (1.0 + q[3] + q[4]);
            z[2 * k + 1] = q[2] * v - q[4] * y;
            z[2 * k]     = q[1] * v - q[3] * y + z[2 * k + 1];
            v = y;
        }
        o->sta[c] = v * v;
        o->lta[c] = v * v;
    }
    o->g = o->lta_len;
    return 0;
}

/*
 * State export / import (NEXT-2; PAPER.md:109 "maintaining correct state propagation", :169 state
 * crosses file boundaries -- here: process boundaries).  out / in: n_ch * (2 n_sec + 2) doubles,
 * per channel z1,z2 of every section, then sta, lta; *g the samples seen.
 */
long long filark_oracle_state_doubles(const filark_oracle_t *o)
{
    return o ? (long long)o->n_ch * (2LL * o->n_sec + 2) : -1;
}
int filark_oracle_get_state(const filark_oracle_t *o, double *out, long long *g)
{
    if (!o || !out || !g) return 1;
    const int w = 2 * o->n_sec + 2;
    for (int c = 0; c < o->n_ch; ++c) {
        memcpy(out + (size_t)c * w, o->z + (size_t)c * 2 * o->n_sec, sizeof(double) * 2 * (size_t)o->n_sec);
        out[(size_t)c * w + 2 * o->n_sec] = o->sta[c];
        out[(size_t)c * w + 2 * o->n_sec + 1] = o->lta[c];
    }
    *g = o->g;
    return 0;
}
int filark_oracle_set_state(filark_oracle_t *o, const double *in, long long g)
{
    if (!o || !in || g < 0) return 1;
    const int w = 2 * o->n_sec + 2;
    for (int c = 0; c < o->n_ch; ++c) {
        memcpy(o->z + (size_t)c * 2 * o->n_sec, in + (size_t)c * w, sizeof(double) * 2 * (size_t)o->n_sec);
        o->sta[c] = in[(size_t)c * w + 2 * o->n_sec];
        o->lta[c] = in[(size_t)c * w + 2 * o->n_sec + 1];
    }
    o->g = g;
    return 0;
}

/*
 * Trigger / event emission on the characteristic function ("any
 * callable that consumes a data window and returns a list of time-channel-bounded events", :132 a
 * threshold-based detector, :169 "must not miss events that straddle two consecutive files").
 * The paper fixes no trigger rule; reading R24: the classic on/off trigger with
 * hysteresis on the float32 CF the path outputs, per channel, state carried across pushes:
 *     off -> on   at the first sample with cf >= thr_on            (t_on = its index, peak = cf)
 *     on  -> off  at the first later sample with cf <  thr_off     (t_off = its index; event emitted)
 *     while on: peak = max(peak, cf)          thr_off <= thr_on, both compared in float32
 * Sample indices count from create/reset.  An event still open when the data end is not emitted
 * (it is, by a later push, when it closes).  Events come out channel by channel in time order.
 */
typedef struct filark_oracle_event {
    long long t_on, t_off;
    int channel;
    float peak;
} filark_oracle_event_t;

typedef struct filark_oracle_trigger {
    int n_ch;
    float thr_on, thr_off;
    int *on;
    long long *t_on;
    float *peak;
    long long g;
} filark_oracle_trigger_t;

filark_oracle_trigger_t *filark_oracle_trigger_create(int n_ch, float thr_on, float thr_off)
{
    if (n_ch <= 0 || !(thr_on > 0.0f) || !(thr_off > 0.0f) || thr_off > thr_on) return NULL;
    filark_oracle_trigger_t *t = (filark_oracle_trigger_t *)calloc(1, sizeof(*t));
    if (!t) return NULL;
    t->n_ch = n_ch; t->thr_on = thr_on; t->thr_off = thr_off;
    t->on = (int *)calloc((size_t)n_ch, sizeof(int));
    t->t_on = (long long *)calloc((size_t)n_ch, sizeof(long long));
    t->peak = (float *)calloc((size_t)n_ch, sizeof(float));
    if (!t->on || !t->t_on || !t->peak) { free(t->on); free(t->t_on); free(t->peak); free(t); return NULL; }
    return t;
}

void filark_oracle_trigger_destroy(filark_oracle_trigger_t *t)
{
    if (!t) return;
    free(t->on); free(t->t_on); free(t->peak); free(t);
}

/* cf: one chunk of the CF, element (c, n) at c*stride_c + n*stride_n.  Appends at most cap events to
 * out; returns the number of events the chunk closed (may exceed cap: the rest is dropped). */
long long filark_oracle_trigger_push(filark_oracle_trigger_t *t, const float *cf, long long n_t,
                                     long long stride_c, long long stride_n,
                                     filark_oracle_event_t *out, long long cap)
{
    if (!t || !cf || n_t < 0) return -1;
    long long n_ev = 0;
    for (int c = 0; c < t->n_ch; ++c) {
        for (long long n = 0; n < n_t; ++n) {
            const float v = cf[(long long)c * stride_c + n * stride_n];
            const long long g = t->g + n;
            if (!t->on[c]) {
                if (v >= t->thr_on) { t->on[c] = 1; t->t_on[c] = g; t->peak[c] = v; }
            } else if (v < t->thr_off) {
                if (out && n_ev < cap) {
                    out[n_ev].t_on = t->t_on[c]; out[n_ev].t_off = g; out[n_ev].channel = c; out[n_ev].peak = t->peak[c];
                }
                n_ev += 1;
                t->on[c] = 0;
            } else if (v > t->peak[c]) {
                t->peak[c] = v;
            }
        }
    }
    t->g += n_t;
    return n_ev;
}

/*
 * Display decimation ("logical downsampling is applied to match
 * the display resolution ... drop mode preserves transient peaks, peak mode maintains amplitude
 * envelopes, and linear interpolation smooths slowly varying wavefields").  The paper gives no
 * formula; reading R25: a window of n_t samples per channel goes to `width` display
 * columns; column j covers the input positions [a_j, a_{j+1}), a_j = floor(j n_t / width)
 * (at least one sample: if a_{j+1} == a_j the column takes sample a_j):
 *     mode 0 "drop":   out[j] = x[a_j]                         (plain striding)
 *     mode 1 "peak":   out[j] = the sample of largest magnitude in the column, the first one on
 *                      ties, with its sign
 *     mode 2 "linear": out[j] = x at position p_j = j (n_t - 1) / (width - 1) (p_0 = 0 for width 1)
 *                      by linear interpolation between the two neighbouring samples, in double
 * Element (c, n) of x at c*stride_c + n*stride_n; out: element (c, j) at c*ostride_c + j*ostride_j.
 */
int filark_oracle_decimate(const float *x, int n_ch, long long n_t, long long stride_c, long long stride_n,
                           int mode, int width, float *out, long long ostride_c, long long ostride_j)
{
    if (!x || !out || n_ch <= 0 || n_t <= 0 || width <= 0 || mode < 0 || mode > 2) return 1;
    for (int c = 0; c < n_ch; ++c) {
        const float *row = x + (long long)c * stride_c;
        for (int j = 0; j < width; ++j) {
            /* floor(j n_t / width) without overflow for the sizes used here (< 2^62) */
            long long a = (long long)j * n_t / width, b = (long long)(j + 1) * n_t / width;
            if (b <= a) b = a + 1;
            if (b > n_t) b = n_t;
            float v;
            if (mode == 0) {
                v = row[a * stride_n];
            } else if (mode == 1) {
                v = row[a * stride_n];
                float best = v < 0.0f ? -v : v;
                for (long long n = a + 1; n < b; ++n) {
                    const float s = row[n * stride_n];
                    const float m = s < 0.0f ? -s : s;
                    if (m > best) { best = m; v = s; }
                }
            } else {
                const double p = width > 1 ? (double)j * (double)(n_t - 1) / (double)(width - 1) : 0.0;
                long long i = (long long)p;
                if (i > n_t - 1) i = n_t - 1;
                const double f = p - (double)i;
                const double x0 = (double)row[i * stride_n];
                const double x1 = (double)row[(i + 1 < n_t ? i + 1 : i) * stride_n];
                v = (float)(x0 + (x1 - x0) * f);
            }
            out[(long long)c * ostride_c + (long long)j * ostride_j] = v;
        }
    }
    return 0;
}

/*
 * Streaming first-order operators ("running automatic gain control
 * (AGC), running mean ... (all with stateful streaming variants)", :122 "gain equalisation (streaming
 * exponential moving average, EMA variant)").  The paper gives no formula; reading R26: the
 * exponential-average forms, state carried across pushes, zero at create/reset:
 *     m[n] = m[n-1] + (u[n] - m[n-1]) / N
 *     mode 0 "running mean":   u = x,    out = m                      (the EMA itself)
 *     mode 1 "de-mean":        u = x,    out = x - m                  (running mean removed)
 *     mode 2 "running AGC":    u = |x|,  out = x / (m + eps)          (gain from the average magnitude)
 */
typedef struct filark_oracle_ema {
    int n_ch, n_len, mode;
    double eps;
    double *m;
} filark_oracle_ema_t;

filark_oracle_ema_t *filark_oracle_ema_create(int n_ch, int n_len, int mode, double eps)
{
    if (n_ch <= 0 || n_len < 1 || mode < 0 || mode > 2 || !(eps >= 0.0)) return NULL;
    filark_oracle_ema_t *o = (filark_oracle_ema_t *)calloc(1, sizeof(*o));
    if (!o) return NULL;
    o->n_ch = n_ch; o->n_len = n_len; o->mode = mode; o->eps = eps;
    o->m = (double *)calloc((size_t)n_ch, sizeof(double));
    if (!o->m) { free(o); return NULL; }
    return o;
}
void filark_oracle_ema_destroy(filark_oracle_ema_t *o) { if (o) { free(o->m); free(o); } }

int filark_oracle_ema_push(filark_oracle_ema_t *o, const float *x, long long n_t, long long stride_c,
                           long long stride_n, float *out)
{
    if (!o || !x || !out || n_t < 0) return 1;
    const double len = (double)o->n_len;
    for (int c = 0; c < o->n_ch; ++c) {
        double m = o->m[c];
        for (long long n = 0; n < n_t; ++n) {
            const long long idx = (long long)c * stride_c + n * stride_n;
            const double v = (double)x[idx];
            const double u = o->mode == 2 ? (v < 0.0 ? -v : v) : v;
            m = m + (u - m) / len;
            out[idx] = (float)(o->mode == 0 ? m : (o->mode == 1 ? v - m : v / (m + o->eps)));
        }
        o->m[c] = m;
    }
    return 0;
}
