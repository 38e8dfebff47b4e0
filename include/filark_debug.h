/*
 * filark_debug.h -- host-only introspection of the preparation stage (no CUDA calls).
 *
 * Used by the CPU test-suite to check the host logic of the library against numpy: the
 * per-section state-space rewrite (s[n] = A s[n-1] + B x[n], y[n] = C s[n-1] + D x[n]) of the
 * SOS operator of PAPER.md:109/121, the float64 block powers the scan relies on, and the
 * tiling of a push of n_t samples.  Return values are filark_status_t codes as int.
 */
#ifndef FILARK_DEBUG_H
#define FILARK_DEBUG_H

#ifdef __cplusplus
extern "C" {
#endif

/*
 * sos    [host, in]  [n_sec][6] doubles (b0 b1 b2 a0 a1 a2).
 * kinds  [host, out] n_sec ints: 0 direct form II, 1 direct form II with explicit b0, 2 delta form,
 *                    3 delta form without a zero at z = 1, 4 normal (coupled) form.  May be NULL.
 * coefs  [host, out] n_sec x 9 doubles: A row-major (4), B (2), C (2), D.  May be NULL.
 * gain   [host, out] product of the b0 factors moved in front of the cascade.  May be NULL.
 * The cascade equals gain * (sections in state-space form applied in order).
 */
int filark_debug_design(const double *sos, int n_sec, int *kinds, double *coefs, double *gain);

/*
 * Slot geometry of one channel-major push of n_t >= 1 samples that finds r0 raw samples of the
 * previous push waiting in the handle (csrc/filark_kernels.cuh): the stream is cut into slots of
 * L samples aligned to the stream (not to the push); a tile is 64 slots (lane l owns slots 2l,
 * 2l+1); tile-space positions [0, r0) of the first tile are the waiting samples.  force_L = 0
 * lets the library choose L among its compiled variants (8, 16, 24), otherwise
 * L = force_L.  out5 = { L, n_tiles, q_last (full slots in the last tile, 0..64), r1 (samples
 * of the trailing partial slot, kept for the next push), vec4 (16-byte accesses stay aligned) }.
 */
int filark_debug_push_geometry(long long n_t, int r0, int force_L, int *out5);

/* out4 (row-major 2x2) = A^e for the state-space form chosen for one section (6 doubles). */
int filark_debug_block_power(const double *sos6, long long e, double *out4);

#ifdef __cplusplus
}
#endif
#endif /* FILARK_DEBUG_H */
