/* fstat.h -- C ABI of the B200-native resampling F-statistic hot path.
 *
 * What it computes: steps (iii)-(vii) of the "Resamp" method of arXiv:2201.00451
 * for a batch of search templates, from the prepared,
 * heterodyned complex64 series x_h(t^k) of each detector (the output
 * of step ii, uploaded once -- PAPER.md:93) to the multi-detector coherent
 * statistic 2F over a frequency band (eq. 8), plus the on-GPU
 * max / top-k retention of PAPER.md:214, :307.
 *
 * Every free choice the paper leaves open (timing model, antenna convention,
 * interpolation kernel, grid placement, normalisation) is fixed in DESIGN.md
 * "Readings"; this header only states argument meaning, layout, ownership and
 * error behaviour.
 *
 * Conventions
 *  - All functions return FSTAT_OK (0) or a negative FSTAT_E* code; no C++
 *    exceptions cross this boundary; no global state.
 *  - "host" pointers are ordinary CPU memory, "device" pointers are CUDA global
 *    memory of the device that was current when fstat_setup ran.
 *  - All GPU work is enqueued on the CUDA stream given to fstat_setup.  Calls
 *    that take device outputs return without waiting for the GPU; host-side
 *    arguments (template arrays) are consumed before the call returns.
 *    Functions with a `_host` suffix block until their host outputs are written.
 *  - One plan must be used from one host thread at a time.
 *  - There is no CPU fallback: without a CUDA device fstat_setup fails with
 *    FSTAT_ECUDA.
 */
#ifndef FSTAT_B200_H
#define FSTAT_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define FSTAT_API __attribute__((visibility("default")))
#else
#define FSTAT_API
#endif

#define FSTAT_OK       0
#define FSTAT_EINVAL  -1   /* bad argument: null pointer, n_det < 1, unsorted / overlapping / off-grid timestamps, k out of range */
#define FSTAT_ESIZE   -2   /* n_fft not a power of two in [2^12, 2^24]; n_samples + 2*ceil(512 s/dt) > n_fft; band > 1/dt; dterms outside [1,32] */
#define FSTAT_EDOM    -3   /* template f0 != plan f_min; antenna determinant D <= 0 (reported by fstat_sync / *_host calls) */
#define FSTAT_ECUDA   -4   /* a CUDA runtime call failed; text via fstat_last_error */
#define FSTAT_ENOMEM  -5   /* host or device allocation failed */

/* Detector site and orientation (S1, S2).  Arms are perpendicular. */
typedef struct {
    double lat_rad;           /* geodetic latitude                                        */
    double lon_east_rad;      /* longitude, east positive                                 */
    double xarm_azimuth_rad;  /* x-arm azimuth, counter-clockwise from local North;
                                 the y-arm is 90 degrees further counter-clockwise         */
} fstat_detector_t;

/* Analytic ephemeris (S3): circular orbit + uniform rotation, Roemer delay
 * only.  All angles are evaluated at t' = t - t_start.  This is t_m(t; alpha, delta)
 * of eq. 3. */
typedef struct {
    double au_over_c_s;    /* orbital radius / c  [s]            */
    double omega_orb;      /* orbital angular rate [rad/s]       */
    double phi_orb0;       /* orbital phase at t_start [rad]     */
    double obliquity_rad;  /* ecliptic obliquity                 */
    double re_over_c_s;    /* Earth radius / c [s]               */
    double omega_rot;      /* sidereal rotation rate [rad/s]     */
    double gmst0_rad;      /* Greenwich sidereal angle at t_start */
} fstat_ephem_t;

/* One search template: the phase parameters lambda of PAPER.md:35, :93.
 * f0 must equal the plan's f_min: one pass computes the whole band;
 * fdot, fddot are the k = 1, 2 coefficients of Phi_s (eq. 3), defined at the SSB
 * reference time tau_ref = t_start (S9). */
typedef struct {
    double alpha;   /* right ascension [rad] */
    double delta;   /* declination [rad]     */
    double f0;      /* [Hz]                  */
    double fdot;    /* [Hz/s]                */
    double fddot;   /* [Hz/s^2]              */
} fstat_template_t;

typedef struct fstat_plan fstat_plan_t;   /* opaque */

/* fstat_setup -- upload the prepared series once and build the plan.
 *
 *  out          receives the plan (caller frees with fstat_destroy).
 *  det[n_det]   host array.
 *  series_c64   host array of n_det pointers; each points to n_samples interleaved
 *               (re, im) float32 pairs = x_h(t_j), t_j = t_start + j*dt, heterodyned at
 *               f_het in the detector frame.  Each pointer may be HOST or DEVICE memory
 *               (detected by the CUDA runtime).  The plan makes its own device copy; the
 *               caller may free or reuse its buffers when fstat_setup returns.
 *               Samples inside gaps must be zero.
 *  timestamps   host array of n_det pointers to n_seg[X] float64 start times of the data
 *               segments ("SFT slots") present for detector X; every entry
 *               must equal t_start + n*t_sft for an integer n >= 0, strictly increasing.
 *  weights      host array of n_det pointers to n_seg[X] float32 noise weights
 *               w = 1/sigma_c^2 of that slot (sigma_c^2: noise variance per real
 *               component of the complex samples; S10, G5).
 *  eph          analytic ephemeris (host).
 *  dterms       D of the windowed-sinc kernel: 2D+1 taps (PAPER.md:83 step v; S6).
 *  f_min, band  the output band [f_min, f_min + band); bin q is f_min + q*df with
 *               df = 1/(n_fft*dt) and n_bins = round(band*n_fft*dt).
 *  n_fft        zero-padded FFT length, a power of two.
 *  cuda_stream  a cudaStream_t (0 = legacy default stream).
 *
 * Device memory owned by the plan: the series (8 B per sample and detector), its Farrow-filtered
 * copies (64 B per sample and detector: the interpolation taps folded once), 8 B per
 * SSB grid point (sidereal-angle table), 32 B per timing node (<= 256 s apart), detector and sky position of a batch, 16 B x n_fft per sky position of a batch (grown on demand, <= 2 GB) and up to
 * 8 GB of FFT intermediates (16 B x n_fft per template of a launch, grown on demand); scratch rows for the top-k and
 * host-output modes on first use.
 */
FSTAT_API int fstat_setup(fstat_plan_t **out, int32_t n_det, const fstat_detector_t *det,
                const void *const *series_c64, int64_t n_samples, double t_start, double dt, double f_het,
                const double *const *timestamps, const float *const *weights, const int32_t *n_seg, double t_sft,
                const fstat_ephem_t *eph, int32_t dterms, double f_min, double band, int64_t n_fft,
                void *cuda_stream);

/* Output layout: 2F[t][q], q in [0, n_bins), is the statistic at f_min + q*df. */
FSTAT_API int fstat_get_layout(const fstat_plan_t *plan, int64_t *n_bins, double *df);

/* fstat_compute -- steps (iii)-(vii) for n_tmpl templates.
 *  tmpl_host   host array; consecutive templates with identical (alpha, delta) share the
 *              sky-dependent work.
 *  twoF_dev    caller-owned DEVICE memory, float32[n_tmpl][n_bins], row-major. */
FSTAT_API int fstat_compute(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, float *twoF_dev);

/* fstat_compute_topk -- same path, but only the k (1..64) loudest bins of every template
 * are kept.  Rows are sorted by descending 2F, ties by ascending bin.
 *  val_dev float32[n_tmpl][k], bin_dev int32[n_tmpl][k]: caller-owned DEVICE memory. */
FSTAT_API int fstat_compute_topk(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, int32_t k,
                       float *val_dev, int32_t *bin_dev);

/* fstat_compute_threshold -- GPU-side candidate retention ("2F > threshold"): for every template
 * the (at most k, 1..64) loudest bins with 2F > threshold, sorted like fstat_compute_topk (unused entries are
 * (-inf, -1)), and the exact number of bins above the threshold (which may exceed k).
 *  val_dev float32[n_tmpl][k], bin_dev int32[n_tmpl][k], count_dev int32[n_tmpl]: caller-owned DEVICE memory.
 *  threshold must be finite (FSTAT_EINVAL otherwise). */
FSTAT_API int fstat_compute_threshold(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, float threshold,
                            int32_t k, float *val_dev, int32_t *bin_dev, int32_t *count_dev);

/* fstat_compute_accumulate -- the semi-coherent building block (section 6: "data ... partitioned into
 * segments ..., each segment is searched using the F-statistic, and results from all segments are summed"): same path
 * as fstat_compute, but 2F is ADDED to what twoF_dev holds, so that the plans of several data segments that share the
 * bin grid (same f_min and df) sum into one array.
 *  bin_offset_host  host int32[n_tmpl] or NULL (= all 0): this plan's bin q of template t is added to output bin
 *                   q - bin_offset[t] (bins that fall outside the row add nothing).  A signal's frequency at this
 *                   segment's reference time tau_ref = t_start differs from its frequency at the search's reference
 *                   time by fdot * (t_start - t_ref) + ...; the caller rounds that to bins.  |offset| < n_bins.
 *  twoF_dev         caller-owned DEVICE memory float32[n_tmpl][n_bins], read and written; the caller zeroes it before the
 *                   first segment.  Calls on the same rows must be ordered on one stream. */
FSTAT_API int fstat_compute_accumulate(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl,
                             const int32_t *bin_offset_host, float *twoF_dev);

/* fstat_compute_per_detector -- the single-detector statistics 2F_X next to the coherent one (the quantity the paper's
 * accuracy tooling compares per detector; eq. 8 with the sums over detector X only):
 *  twoF_dev   caller-owned DEVICE memory float32[n_det][n_tmpl][n_bins].
 * A detector without valid data gives D_X <= 0: its rows are NaN and fstat_sync reports FSTAT_EDOM. */
FSTAT_API int fstat_compute_per_detector(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, float *twoF_dev);

/* fstat_select_topk / fstat_select_threshold -- the selection of fstat_compute_topk / fstat_compute_threshold applied to
 * rows the caller already holds in DEVICE memory (float32[n_rows][n_bins] of this plan's bin layout), e.g. the summed 2F
 * of a semi-coherent search (PAPER.md:325 with the retention of PAPER.md:307).  Same ordering, tie rule and outputs. */
FSTAT_API int fstat_select_topk(fstat_plan_t *plan, const float *twoF_dev, int32_t n_rows, int32_t k, float *val_dev, int32_t *bin_dev);
FSTAT_API int fstat_select_threshold(fstat_plan_t *plan, const float *twoF_dev, int32_t n_rows, float threshold, int32_t k,
                           float *val_dev, int32_t *bin_dev, int32_t *count_dev);

/* fstat_select_topk_noalloc -- fstat_select_topk for callers that must not allocate device memory.
 *
 * Who needs it.  Two kinds of caller cannot let this library call cudaMalloc on their behalf:
 *  (1) a search pipeline that has handed the whole GPU to its own arena or pool at start-up (the summed 2F rows of a
 *      semi-coherent search, are typically held in such an arena): nothing is left for cudaMalloc to
 *      give, so the plan-based calls, which create their scratch on first use, fail with an allocation error;
 *  (2) a follow-up stage inside a latency-bound loop: cudaMalloc and cudaFree synchronise the whole device and stall
 *      every other stream while they run.
 * This call needs no plan (fstat_setup allocates) and calls no cudaMalloc, cudaFree or other allocating routine.  Its
 * only scratch -- one uint32 maximum per group of 512 bins, the table the selection kernel reads to find the groups
 * that can hold a top-k bin -- is a fixed array of FSTAT_NOALLOC_MAX_GROUPS entries (1 MiB) inside the library image.
 * Every GPU that loads the library carries that 1 MiB until the process exits, whether or not this call is used.
 *
 *  twoF_dev   caller-owned DEVICE memory float32[n_rows][n_bins], row-major, read only.
 *  n_bins     1 .. 2^24 bins per row (any value: rows need not be a multiple of 512).
 *  n_rows     >= 0;  n_rows * ceil(n_bins / 512) must not exceed FSTAT_NOALLOC_MAX_GROUPS: e.g. 64 rows of 2^22 bins
 *             or 4096 rows of 2^16 bins per call.  Larger requests are rejected with FSTAT_ESIZE and nothing is
 *             launched; split them over several calls on the same stream.
 *  k          1 .. min(64, n_bins).
 *  val_dev float32[n_rows][k], bin_dev int32[n_rows][k]: caller-owned DEVICE memory; same order, tie rule and values
 *             (bit for bit) as fstat_select_topk.
 *  cuda_stream  a cudaStream_t (0 = legacy default stream); the call returns without waiting for the GPU.
 *
 * The device that holds the rows must be current.  The FIRST call on each device does a one-time set-up (it looks up
 * the device address of the scratch array and raises the selection kernel's shared-memory limit); make that first call
 * before any stream capture begins.  All calls on a device share the one array and it keeps whatever the last call
 * left in it: the call overwrites every entry it reads, so nothing has to be cleared, but two calls whose GPU work
 * overlaps (different streams, different host threads) race on it -- keep them on one stream or order them with
 * events.  Errors: FSTAT_EINVAL (null pointer, k out of range, n_rows < 0), FSTAT_ESIZE (limits above), FSTAT_ECUDA;
 * the text is available from fstat_last_error(NULL) on the calling thread. */
#define FSTAT_NOALLOC_MAX_GROUPS 262144
FSTAT_API int fstat_select_topk_noalloc(const float *twoF_dev, int64_t n_bins, int32_t n_rows, int32_t k,
                              float *val_dev, int32_t *bin_dev, void *cuda_stream);

/* Host-buffer variants (the end-to-end entry points): outputs are HOST memory (pinned
 * memory makes the copies asynchronous and overlapped); they return after the data
 * has landed and report FSTAT_EDOM if a template had D <= 0. */
FSTAT_API int fstat_compute_host(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, float *twoF_host);
FSTAT_API int fstat_compute_topk_host(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, int32_t k,
                            float *val_host, int32_t *bin_host);

/* fstat_resample_sky -- the sky-dependent half of the path on its own (steps iii-v and the
 * a, b weighting of step vi): writes the detector-summed, resampled series
 *   S[k] = ( Re Ya0, Im Ya0, Re Yb0, Im Yb0 ),  k in [0, n_fft)  (zero beyond the data),
 * i.e. Fa(t), Fb(t) before the spin-down factor, already shifted so that FFT index q is
 * output bin q, into caller-owned DEVICE memory float32[n_fft][4]; and the antenna sums
 * A, B, C, D = AB - C^2 (eq. 8) into HOST abcd[4] (this call synchronises the stream). */
FSTAT_API int fstat_resample_sky(fstat_plan_t *plan, double alpha, double delta, float *S_dev, double *abcd_host);

/* Wait for all work enqueued by this plan; returns FSTAT_EDOM if any template since the
 * last sync had D <= 0 (its outputs are NaN), FSTAT_ECUDA on a device fault. */
FSTAT_API int fstat_sync(fstat_plan_t *plan);

/* Measurement and experiment hooks (launch counter, per-kernel-class timing, launch-shape overrides) are declared in
 * fstat_debug.h; nothing on the product path needs them. */

FSTAT_API void fstat_destroy(fstat_plan_t *plan);

FSTAT_API const char *fstat_strerror(int code);
/* Text of the last error on this plan (includes the CUDA error string for FSTAT_ECUDA).
 * The pointer stays valid until the next failing call on the plan. plan may be NULL
 * to query the last fstat_setup failure of the calling thread. */
FSTAT_API const char *fstat_last_error(const fstat_plan_t *plan);

#ifdef __cplusplus
}
#endif
#endif /* FSTAT_B200_H */
