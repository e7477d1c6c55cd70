/* fstat_debug.h -- measurement and experiment hooks of the B200 F-statistic library.
 *
 * Not part of the computation ABI (fstat.h): nothing here changes what is computed, only how the work is
 * launched or what is recorded about it.  bench.py uses the launch counter and the per-class timing for its
 * roofline report; the tests use the launch-shape overrides to reach every kernel variant
 * and the multi-batch paths at small sizes.  Same conventions as fstat.h (FSTAT_OK or a negative FSTAT_E* code).
 */
#ifndef FSTAT_B200_DEBUG_H
#define FSTAT_B200_DEBUG_H

#include "fstat.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Number of kernels this plan has launched since setup (bench.py's `gpu_launches`). */
FSTAT_API int fstat_launch_count(const fstat_plan_t *plan, int64_t *count);

/* How many templates' four-step intermediates are kept in flight per launch (0 = the plan's default, which depends on
 * n_fft, the SM count and the device's memory; 1 .. FSTAT_MAX_INFLIGHT otherwise, FSTAT_EINVAL beyond); bounds the
 * L2 / HBM footprint of the FFT (16 B x n_fft per template, allocated on demand). */
#define FSTAT_MAX_INFLIGHT 65536
FSTAT_API int fstat_set_inflight(fstat_plan_t *plan, int32_t n_inflight);

/* Per-kernel-class device timing with CUDA events on the plan's stream (for the roofline report,
 * SURVEY.md 8(d)).  While enabled, every group of launches of one class is bracketed by two events.
 * fstat_get_profile waits for the stream, writes the summed elapsed milliseconds and launch counts since
 * the last call into HOST ms[FSTAT_PROFILE_CLASSES], launches[FSTAT_PROFILE_CLASSES], and resets the record.
 * Classes: 0 = sky-dependent kernels (timing, resampling), 1 = FFT pass 1 (spin-down prologue + column
 * FFTs), 2 = FFT pass 2 (row FFTs + 2F epilogue), 3 = top-k, 4 = fused sky + pass 1 (sky-varying search),
 * 5 = single-kernel FFT (small n_fft). */
#define FSTAT_PROFILE_CLASSES 6
FSTAT_API int fstat_set_profile(fstat_plan_t *plan, int32_t enable);
FSTAT_API int fstat_get_profile(fstat_plan_t *plan, double *ms, int64_t *launches);

/* Launch-shape override for experiments and tests: n_fft = 2^log_n1 x 2^log_n2 with pass 2 transforming
 * 2^log_n2 points, tiles of 2^log_tile1 / 2^log_tile2 elements, p2_elems (16 or 32) register elements per
 * pass-2 thread.  Any argument < 0 keeps the plan's default for that field.  FSTAT_ESIZE if no kernel is
 * instantiated for the combination (the plan is left unchanged).  Results do not depend on the shape beyond
 * fp32 rounding order. */
FSTAT_API int fstat_debug_set_geometry(fstat_plan_t *plan, int32_t log_n2, int32_t log_tile1, int32_t log_tile2, int32_t p2_elems);

/* Upper bound on the sky positions resampled per batch (default: 2 GB of resampled series); lets a test reach
 * the multi-batch path with a handful of sky positions.  0 = default. */
FSTAT_API int fstat_debug_set_max_sky_slots(fstat_plan_t *plan, int32_t max_slots);

/* Which path serves sky-varying banks / small FFTs: -1 = automatic (default), 0 = off, 1 = forced where supported.
 *   fused_sky : per-sky work (H1-H5) inside the FFT pass-1 prologue instead of the hoisted sky kernel + S buffer
 *               (PAPER.md:188, :293 sky-varying searches); needs pass 1 on tiles of >= 2^11 elements
 *               (fstat_debug_set_geometry(-1, 11, -1, -1) where the default is the one-warp 2^10-element tile).
 *               Automatic = off: measured slower on B200.
 *   single    : one cooperative kernel for both FFT passes of groups of templates whose four-step intermediate
 *               stays in L2 (n_fft <= 2^18, both passes on 2^11-element tiles and one of the splits 2^6 x 2^6, 2^7 x 2^6, 2^7 x 2^7,
 *               2^9 x 2^6, 2^10 x 2^6 / 2^7 / 2^8: e.g. fstat_debug_set_geometry(6, 11, 11, -1) at n_fft = 2^16).
 *               Automatic = off: measured never faster than the two-launch form on B200. */
FSTAT_API int fstat_debug_set_paths(fstat_plan_t *plan, int32_t fused_sky, int32_t single);

/* fstat_debug_compute_fafb -- the path of fstat_compute, but the pass-2 epilogue stores the two spectra instead of
 * combining them with eq. 8: the paper's accuracy tooling compares "the output for F, Fa, and Fb" (Fig. 4),
 * and 2F alone cannot see a slip that leaves the quadratic form unchanged (Fa <-> conj Fa, a common phase).
 *  fafb_dev  caller-owned DEVICE memory float32[n_tmpl][n_bins][4] = (Re Fa, Im Fa, Re Fb, Im Fb) of bin q = f_min + q df,
 *            on the grid convention of DESIGN.md S7 (SSB grid index 0 at t_start - K_m dt: compare with another
 *            implementation only up to the common factor exp(+2 pi i (f - f_het) K_m dt)).
 * For accuracy checks on small banks: 16 B per bin, and only for the default launch shapes of n_fft <= 2^22
 * (FSTAT_ESIZE otherwise). */
FSTAT_API int fstat_debug_compute_fafb(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, float *fafb_dev);

#ifdef __cplusplus
}
#endif
#endif /* FSTAT_B200_DEBUG_H */
