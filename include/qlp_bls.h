/*
 * qlp_bls.h -- C ABI of the B200-native QLP transit-search hot path.
 *
 * What it computes: the Box Least Squares spectrum (Kovacs et al. 2002; named as the search
 * algorithm at) of many ragged TESS light curves over a per-star Keplerian
 * frequency / duration grid, the paper's S/N spectrum (PAPER.md:37-42,
 * Eq. 1 and footnote 3 at :65) and the top peaks.  Paper = arXiv:2302.01293,
 * "QLP Data Release Notes 003: GPU-based Transit Search".  Where the paper is silent the readings
 * of DESIGN.md ("Readings", A1..A26) apply; the step names S0..S4 / O0..O6 are DESIGN.md's.
 *
 * Conventions for every entry point
 *   - "dev" pointers are CUDA device memory on the context's device, "host" pointers are host
 *     memory.  All arrays are caller-owned; the library reads inputs, writes outputs and keeps no
 *     pointer after the call returns.  The context owns only its own workspace.
 *   - Work is enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL = default stream).
 *     Only qlp_bls_grid() synchronises the stream (to return two totals to the host).
 *   - Return value: 0 on success, negative qlp_bls_status otherwise.  No exceptions, no aborts,
 *     nothing written to stdout/stderr.  Data-dependent degeneracy is not an error: a star with
 *     fewer than two points, zero baseline or P_max <= P_min gets grid.status != 0, n_freq = 0 and
 *     empty outputs.
 *   - A context is not thread-safe; use one per host thread / stream.
 *   - Layout: ragged CSR over stars.  Points: row_ptr[S+1] (int64), star s owns
 *     [row_ptr[s], row_ptr[s+1]).  Frequencies: freq_ptr[S+1] (int64), ascending frequency within
 *     a star.  t in days (any zero point), strictly increasing within a star; y any linear flux
 *     unit; dy > 0.  rho in solar units (non-finite or <= 0 means "solar").
 *     The weights dy^-2 / sum dy^-2 are accumulated in 32-bit fixed point (resolution 2^-32 of a star's total
 *     weight): the SR tolerance of 1e-4 of the peak holds for errors that vary by less than a factor ~30 within one
 *     light curve; beyond that, boxes made of a few very light points are resolved to a few 1e-4.
 */
#ifndef QLP_BLS_H_
#define QLP_BLS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qlp_bls_ctx qlp_bls_ctx; /* opaque, owned by the library */

enum qlp_bls_status {
  QLP_BLS_OK = 0,
  QLP_BLS_EINVAL = -1,       /* NULL pointer, negative size, bad config field                   */
  QLP_BLS_ENOMEM = -2,       /* workspace allocation failed                                      */
  QLP_BLS_ECUDA = -3,        /* a CUDA runtime call or kernel launch failed                      */
  QLP_BLS_EUNSUPPORTED = -4, /* e.g. a star needs more phase bins than QLP_BLS_MAX_NB            */
  QLP_BLS_EVALIDATION = -5,  /* flags bit0 set and an input failed validation                    */
  QLP_BLS_ETOOLARGE = -6     /* qlp_bls_grid_noalloc: n_stars > QLP_BLS_NOALLOC_MAX_STARS        */
};

/* Largest number of fine phase bins per frequency (two FP32 histograms of one frequency must fit
 * one SM's shared memory; reading A16).  Not reached for rho* <= 30, P <= 180 d. */
#define QLP_BLS_MAX_NB 24576

/* Largest number of points per star (the 32-bit fixed-point weights of the shared-memory histograms must not
 * overflow when every point of a star lands in one bin).  Longer light curves are skipped with status 5. */
#define QLP_BLS_MAX_POINTS 4194304

/* Search parameters.  POD, caller-owned, copied by qlp_bls_create().  Defaults = the paper's. */
typedef struct {
  uint32_t struct_bytes;    /* = sizeof(qlp_bls_config), for versioning                          */
  int32_t device;           /* CUDA device ordinal                                               */
  double samples_per_peak;  /* 2.0                                                 */
  double dlogq;             /* 0.1                                                 */
  int32_t noverlap;         /* 3                                                 */
  int32_t top_k;            /* peaks reported per star, 1..8                                     */
  double qmin_fac;          /* 0.5   PAPER.md:19 ("between 0.5 and 2.0 times" the circular one)  */
  double qmax_fac;          /* 2.0                                                 */
  double a_over_rstar_min;  /* 2.0 (3.0 = the Sectors 59-60 variant)                */
  double sector_days;       /* 27.4                                                  */
  uint32_t flags;           /* bit0: validate inputs on the device (t finite and strictly
                               increasing in qlp_bls_grid; y, dy finite and dy > 0 in
                               qlp_bls_spectrum, which then synchronises once); a violation makes
                               the call return QLP_BLS_EVALIDATION.
                               bit1: the comparison grid has equal steps in FREQUENCY (see below;
                               read by qlp_bls_grid only).  Other bits reserved: qlp_bls_create
                               returns QLP_BLS_EINVAL unless they (and reserved_) are 0            */
  uint32_t reserved_;       /* 0                                                                 */
  /* Comparison grid (O1.10; the earlier CPU search used "an under-sampled
   * frequency grid on the order of 80,000 frequencies or less" and "periods up to only ~56 days").
   * Both 0 (default) = the paper's GPU grid.  Only qlp_bls_grid reads them.  qlp_bls_create returns
   * QLP_BLS_EINVAL for max_period_days < 0 (or NaN), max_freq < 0 or max_freq == 1.
   * flags bit1 (O1.10c; "uniform <= 80,000-frequency grid, P <= 56 d"): f_k = f_min + k df
   * over the same range [1 / p_max, 1 / p_min] instead of equal steps in f^(1/3); df = the step of the f^(1/3) law
   * at f_min (its finest), or (f_max - f_min) / (max_freq - 1) when that takes more than max_freq points.  nb_k
   * keeps the Keplerian law at f_k.  A star whose step would be below 1e-9 f_max gets status 3.                */
  double max_period_days;   /* > 0: P_max = min(P_max, max_period_days)                          */
  int64_t max_freq;         /* >= 2: a star whose grid has more frequencies gets exactly max_freq
                               of them over the same range, step (u1 - u0) / (max_freq - 1)      */
} qlp_bls_config;

/* Per-star grid descriptor, written by qlp_bls_grid() (device memory, one per star).
 * Frequency k of the star is f_k = u^3 with u = u0 + k*h (FP64, in that order), and its number
 * of fine phase bins is nb_k = ceil(noverlap / (qmin_fac * c_q * u^2)).  DESIGN.md O1.
 * On the frequency-uniform comparison grid (flags bit1) h is NEGATIVE and marks the kind of grid:
 * f_k = u0 + k*(-h) with u0 = 1 / p_max, and nb_k by the same formula with u = cbrt_det(f_k). */
typedef struct {
  double t_ref;     /* first timestamp: phase zero point (reading A4)                            */
  double baseline;  /* T = t_last - t_first, days                                                */
  double p_min;     /* period at which a = a_over_rstar_min * R*   PAPER.md:23                    */
  double p_max;     /* longest continuous stretch, or half of it                    */
  double c_q;       /* q_circ(f) = c_q * f^(2/3)                    */
  double u0;        /* cbrt_det(1 / p_max)   (flags bit1: 1 / p_max)                             */
  double h;         /* grid step in u = f^(1/3)                    PAPER.md:35 (samples_per_peak)
                       (flags bit1: minus the step in frequency)                                 */
  int64_t n_freq;   /* number of trial frequencies                                               */
  int32_t nb_max;   /* phase bins at k = 0 (the largest)                                         */
  int32_t status;   /* 0 ok; 1 fewer than 2 points; 2 baseline <= 0; 3 f_max <= f_min (or, flags
                       bit1, a frequency step below 1e-9 f_max);
                       4 nb_max > QLP_BLS_MAX_NB (star skipped, n_freq = 0);
                       5 more than QLP_BLS_MAX_POINTS points (star skipped, n_freq = 0);
                       7 timestamps not finite and strictly increasing (star skipped, n_freq = 0:
                         checked for every star, whether or not flags bit0 asks for validation)    */
} qlp_bls_star_grid;

/* One peak of one star, written by qlp_bls_snr() (device memory, [S * top_k], rank-major within
 * a star).  Unused slots have k = -1, status = 1.  PAPER.md:44 (period, epoch, depth, duration
 * are what the next pipeline stage takes from the BLS). */
typedef struct {
  int64_t k;       /* frequency index within the star's grid                                     */
  double freq;     /* d^-1                                                                       */
  double period;   /* d                                                                          */
  double t0;       /* mid-transit epoch, same zero point as t                                    */
  float sr;        /* SR at k                                                                    */
  float snr;       /* S/N at k  (Eq. 1)                                          */
  float q;         /* m / nb : best duty cycle                                                   */
  float depth;     /* -s / (r (1 - r)): positive for a dip                                       */
  int32_t m;       /* best box width in fine bins                                                */
  int32_t j;       /* best box start bin                                                         */
  int32_t nb;      /* fine bins at k                                                             */
  int32_t status;  /* 0 = valid                                                                  */
} qlp_bls_peak;

/* "Other statistics" of one peak, written by qlp_bls_peak_stats() (device memory, [S * top_k],
 * same order as the peak table).  DESIGN.md O7: a point is in transit when it lies within half a duration of the
 * nearest expected mid-transit time T0 + n P, "before" / "after" are the one-duration-wide windows next to the
 * transit, a transit counts only if it owns at least one in-transit point, and the out-of-transit level is the
 * dy^-2-weighted mean of y over the points that are not in transit.  Invalid peaks give all zeros. */
typedef struct {
  int32_t n_in;        /* points in transit (n_t of PAPER.md Eq. 2)                                */
  int32_t n_before;    /* points in [-1.5 D, -0.5 D) around the mid-times                          */
  int32_t n_after;     /* points in (0.5 D, 1.5 D]                                                  */
  int32_t n_transits;  /* transits with data within 0.5 D of the mid-time (N_t of PAPER.md Eq. 2)  */
  double oot_level;    /* out-of-transit level, same unit as y                                     */
  double duration;     /* D = (m / nb) * period, days                                              */
} qlp_bls_transit_stats;

/* Trapezoid fit of one peak, written by qlp_bls_trapezoid_fit() (device memory, [S * top_k], same
 * order as the peak table).  DESIGN.md O8: model y ~ z - depth * sh(|dt - (t0 - t0_bls)|) with sh the unit trapezoid
 * of total duration q P and ingress q_in q P; P = 1/freq stays fixed; the data are the points within two BLS
 * durations of the BLS mid-transit times.  status: 0 fitted, 1 no peak (all fields of the start point), 2 fewer than
 * 5 points in the window (not fitted: t0, q of the BLS, q_in = 0.25). */
typedef struct {
  double t0;          /* transit epoch (same zero point as t)                                       */
  double depth;       /* > 0 for a dip of y (sign convention of qlp_bls_peak.depth)                 */
  double q;           /* duration / period, in [0, 1]                                               */
  double q_in;        /* ingress duration / duration, in [0, 0.5]                                   */
  double z;           /* out-of-transit level, unit of y                                            */
  double chi2;        /* sum dy^-2 (y - model)^2 over the fitted points                             */
  double chi2_init;   /* the same at the start point (t0_bls, q_bls, 0.25)                          */
  int32_t n_fit;      /* points in the window                                                       */
  int32_t n_eval;     /* chi2 evaluations spent (no sweep of six starts after 600)                  */
  int32_t status;
  int32_t pad_;
} qlp_bls_trapezoid;

/* Noise estimates, signal-to-pink-noise and detection flag of one peak (PAPER.md:45-51 with Eq. 2, :55), written by
 * qlp_bls_pink_noise() (device memory, [S * top_k], same order as the peak table).  DESIGN.md O9: residuals of all
 * points of the star against the fitted trapezoid; sigma_w = their rms about the mean; sigma_r^2 = variance of the
 * means over time bins of one transit duration minus sigma_w^2 mean(1/n_b), floored at 0; S/N_pink = depth_eff /
 * sqrt(sigma_w^2 / n_t + sigma_r^2 / n_transits).  Peaks without a fit (fit status != 0) give all zeros. */
typedef struct {
  double sigma_w;      /* white noise, unit of y                                                     */
  double sigma_r;      /* red noise on the timescale of the fitted duration                          */
  double depth_eff;    /* depth (1 - q_in): the trapezoid integral over the duration   */
  double snr_pink;     /* PAPER.md Eq. 2 with depth_eff                                              */
  int32_t n_t;         /* points in transit (fitted epoch and duration)                              */
  int32_t n_transits;  /* transits with data within 0.5 durations of mid-transit                     */
  int32_t n_bins;      /* non-empty duration-long time bins                                          */
  int32_t detected;    /* 1 iff n_transits >= 2, snr_pink > 9 and the peak's S/N > 9    */
} qlp_bls_pink;

/* Fill *cfg with the paper's defaults, device 0, top_k 3. */
void qlp_bls_default_config(qlp_bls_config* cfg /*host*/);

/* Create a context on cfg->device.  Returns EINVAL for out-of-range fields (noverlap < 1,
 * widths not inside [1, 31], top_k outside 1..8, non-positive factors), ECUDA if the device
 * cannot be used. */
int qlp_bls_create(const qlp_bls_config* cfg /*host*/, qlp_bls_ctx** out /*host*/);

/* S1, per-star Keplerian grid (O1).
 *   in : row_ptr dev int64[S+1]; t dev double[row_ptr[S]]; rho, rstar dev double[S]
 *        (rstar may be NULL: it cancels, reading A8).
 *   out: grid dev [S]; freq_ptr dev int64[S+1] (exclusive scan of n_freq);
 *        *total_freq = freq_ptr[S] and *total_bins = sum over all frequencies of nb_k (host).
 * Synchronises the stream. */
int qlp_bls_grid(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                 const double* rho, const double* rstar, qlp_bls_star_grid* grid, int64_t* freq_ptr,
                 int64_t* total_freq, int64_t* total_bins, void* cuda_stream);

/* S1 for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): the same two kernels as qlp_bls_grid (O1), same grid
 * descriptors and freq_ptr bit for bit, but the stage's scratch array (one 64-bit sum of nb_k per star) is a
 * file-scope __device__ array of the library instead of context workspace, and the two totals stay on the device.
 * The call makes no cudaMalloc / cudaFree / allocating library call, copies nothing to the host and does not
 * synchronise: it enqueues one memset of the used scratch prefix and two kernels on `cuda_stream`.
 *   in : row_ptr dev int64[S+1]; t dev double[row_ptr[S]]; rho dev double[S]
 *   out: grid dev [S]; freq_ptr dev int64[S+1]; totals dev int64[2] = { freq_ptr[S], sum of nb_k }.
 * Limits and contract:
 *   - n_stars <= QLP_BLS_NOALLOC_MAX_STARS (262,144; the static array is 2 MiB, held by every GPU that loads the
 *     library until the process exits); a larger batch returns QLP_BLS_ETOOLARGE and enqueues nothing;
 *   - no input validation pass, whatever flags bit0 says (it needs a read-back); stars with non-increasing or
 *     non-finite timestamps still get status 7 and n_freq = 0 as in qlp_bls_grid;
 *   - ALL calls on a device share the one array, and it keeps the last call's contents: two calls that may overlap
 *     on the GPU (different streams, different contexts, different host threads) race on it.  Serialise them
 *     (one stream, or an event between them);
 *   - the first call on a device resolves the array's device address (cudaGetSymbolAddress, once per device): make
 *     one call before starting a graph capture.
 * `ctx` supplies the search parameters and the device; its workspace is not touched. */
#define QLP_BLS_NOALLOC_MAX_STARS 262144
int qlp_bls_grid_noalloc(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                         const double* rho, qlp_bls_star_grid* grid, int64_t* freq_ptr, int64_t* totals,
                         void* cuda_stream);

/* S0 + S2 + S3: weights and centred series (Kovacs 2002 weighting), fold-and-bin
 * at every grid frequency, box scan over every start bin and every width of the duration ladder
 * (PAPER.md:19, :35).  DESIGN.md O2-O4.
 *   in : as qlp_bls_grid plus y, dy dev double[row_ptr[S]], and grid / freq_ptr from qlp_bls_grid.
 *   out: sr dev float[total_freq]   SR(f) = max over boxes of s^2 / (r (1 - r));
 *        best dev uint32[total_freq] = (m << 24) | j  of the maximising box. */
int qlp_bls_spectrum(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                     const double* y, const double* dy, const qlp_bls_star_grid* grid,
                     const int64_t* freq_ptr, float* sr, uint32_t* best, void* cuda_stream);

/* S4: the paper's S/N spectrum (median-binned trend, interpolated and subtracted,
 * sigma = 1.4826 MAD; bin count by Sturges' law, footnote 3 at :65) and the top_k peaks with
 * period, epoch, depth, duration.  DESIGN.md O5-O6.
 *   in : as qlp_bls_spectrum plus its outputs sr, best.
 *   out: snr dev float[total_freq] or NULL; peaks dev [S * top_k].
 * The prepared point records of the last qlp_bls_spectrum call of this context are reused when this call names
 * the same arrays (row_ptr, t, y, dy, grid pointers and n_stars) and no other call of the context touched the
 * workspace in between; otherwise S0 is run again.  The caller must not rewrite those arrays in place between
 * the two calls. */
int qlp_bls_snr(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                const double* y, const double* dy, const qlp_bls_star_grid* grid,
                const int64_t* freq_ptr, const float* sr, const uint32_t* best, float* snr,
                qlp_bls_peak* peaks, void* cuda_stream);

/* Per-peak statistics (O7; the row after the search in SURVEY.md 8(f)).
 *   in : the batch (row_ptr, t, y, dy) and the peak table written by qlp_bls_snr, all dev.
 *   out: stats dev [S * top_k]. */
int qlp_bls_peak_stats(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t, const double* y,
                       const double* dy, const qlp_bls_peak* peaks, qlp_bls_transit_stats* stats, void* cuda_stream);

/* Trapezoid fit of every peak (O8): epoch, depth, q, q_in and level by
 * least squares at the fixed BLS period, from the BLS values, on the points within two durations of mid-transit.
 *   in : the batch (row_ptr, t, y, dy) and the peak table written by qlp_bls_snr, all dev.
 *   out: fits dev [S * top_k].
 * Synchronises the stream once (the workspace is sized from the number of points inside the fit windows).
 * Returns EUNSUPPORTED if one window holds 2^31 points or more. */
int qlp_bls_trapezoid_fit(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t, const double* y,
                          const double* dy, const qlp_bls_peak* peaks, qlp_bls_trapezoid* fits, void* cuda_stream);

/* Noise estimates, S/N_pink and the detection criteria of every peak (O9; SURVEY.md
 * 8(f) f3).
 *   in : the batch (row_ptr, t, y), the peak table of qlp_bls_snr and the fits of qlp_bls_trapezoid_fit, all dev.
 *   out: pink dev [S * top_k].  Asynchronous on the stream. */
int qlp_bls_pink_noise(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t, const double* y,
                       const qlp_bls_peak* peaks, const qlp_bls_trapezoid* fits, qlp_bls_pink* pink, void* cuda_stream);

/* Whole path with HOST buffers (pageable or pinned): copies the batch to the device in sub-batches (the copy of
 * the next one overlaps the search of the current one), runs grid -> spectrum -> snr (-> peak_stats), copies the
 * peak table (and the statistics) back.  This is the call the end-to-end benchmark times.
 * peaks host [S * top_k]; stats host [S * top_k] or NULL; grid_out host [S] or NULL; total_freq host or NULL. */
int qlp_bls_search_host(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                        const double* y, const double* dy, const double* rho, const double* rstar,
                        qlp_bls_peak* peaks, qlp_bls_transit_stats* stats, qlp_bls_star_grid* grid_out,
                        int64_t* total_freq, void* cuda_stream);

/* qlp_bls_search_host followed, per sub-batch, by the rows after the search: trapezoid fit and noise /
 * S/N_pink / detection flag, also copied back.  fits host [S * top_k] or NULL; pink host [S * top_k]
 * or NULL (pink needs the fits on the device, they are computed even if fits is NULL).  Everything else as
 * qlp_bls_search_host. */
int qlp_bls_vet_host(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t, const double* y,
                     const double* dy, const double* rho, const double* rstar, qlp_bls_peak* peaks,
                     qlp_bls_transit_stats* stats, qlp_bls_trapezoid* fits, qlp_bls_pink* pink,
                     qlp_bls_star_grid* grid_out, int64_t* total_freq, void* cuda_stream);

/* Release the context and its workspace.  NULL is allowed. */
int qlp_bls_destroy(qlp_bls_ctx* ctx);

/* Static string for a status code. */
const char* qlp_bls_strerror(int code);

/* Number of kernels this context has launched since creation (bench.py's gpu_launches). */
int64_t qlp_bls_launch_count(const qlp_bls_ctx* ctx);

/* CUDA-event timing of the fold/scan launches inside qlp_bls_spectrum (the dominant kernel; used by
 * bench.py for the roofline figure).  enable != 0 starts recording one event pair per spectrum call
 * on the call's stream (a ring of 256) and resets the call count. */
int qlp_bls_fold_timing(qlp_bls_ctx* ctx, int32_t enable);

/* Waits for the recorded events; *n_calls = spectrum calls timed (<= 256), *total_ms = summed device
 * time of their fold/scan launches. */
int qlp_bls_fold_elapsed_ms(qlp_bls_ctx* ctx, int32_t* n_calls /*host*/, double* total_ms /*host*/);

/* While fold timing is on, the fold/scan kernel also adds up thread 0's SM clocks per phase over all tiles:
 * clocks[0] = tile set-up + zeroing, clocks[1] = fold (S2), clocks[2] = box scan + reduction + output (S3).
 * Their ratios split the fused kernel's time between S2 and S3.  Synchronises the device.  clocks host [3]. */
int qlp_bls_fold_phase_clocks(qlp_bls_ctx* ctx, uint64_t* clocks /*host*/);

/* Work of the trapezoid fits since qlp_bls_fold_timing(ctx, 1): out host uint64[2], out[0] = (point, sweep) pairs in
 * which the point lay inside some candidate's transit (each is six trapezoid evaluations of O8), out[1] reserved.
 * Synchronises the device. */
int qlp_bls_fit_work(qlp_bls_ctx* ctx, uint64_t* out);

/* Per tile class c = 0..8 of the fold/scan kernel, summed over all tiles since
 * qlp_bls_fold_timing(ctx, 1): out host uint64[9][5] = {set-up + zeroing clocks, fold clocks, scan clocks (SM clocks
 * of thread 0 of each CTA), point x frequency evaluations, tiles}.  Synchronises the device. */
int qlp_bls_fold_class_counters(qlp_bls_ctx* ctx, uint64_t* out);

/* The duration ladder in fine bins (O1.9): writes up to cap widths to m (host),
 * returns their number. */
int qlp_bls_widths(const qlp_bls_ctx* ctx, int32_t* m /*host*/, int32_t cap);

/* ---- test-only entry points (parity tests call them through the same ABI) ---- */

/* f_k and nb_k for k in [k0, k1) of one star.  grid dev [S]; f dev double[k1-k0]; nb dev int32[k1-k0]. */
int qlp_bls_debug_freqs(qlp_bls_ctx* ctx, const qlp_bls_star_grid* grid, int64_t star, int64_t k0,
                        int64_t k1, double* f, int32_t* nb, void* cuda_stream);

/* Bin index (O3) of every point of one star at grid frequency k, computed with the same
 * device function the fold kernels use.  bin_of_point dev int32[N_star]. */
int qlp_bls_debug_bins(qlp_bls_ctx* ctx, const int64_t* row_ptr, const double* t,
                       const qlp_bls_star_grid* grid, int64_t star, int64_t k, int32_t* bin_of_point,
                       void* cuda_stream);

/* S0 outputs of one star: tau dev double[N], w dev float[N], wy dev float[N]. */
int qlp_bls_debug_prep(qlp_bls_ctx* ctx, const int64_t* row_ptr, const double* t, const double* y,
                       const double* dy, const qlp_bls_star_grid* grid, int64_t star, double* tau,
                       float* w, float* wy, void* cuda_stream);

/* Bounds-check build only (`python -m paper_2302_01293_b200.build --check` -> libqlp_bls_check.so, compiled with
 * -DQLP_BOUNDS_CHECK): every guarded shared-memory / workspace access of the fold, scan and fit kernels tests its index
 * against the extent it must stay in and counts a violation instead of performing the access.  out host uint64[8]:
 * [0] fold histogram cell, [1] staging chunk, [2] scan bin, [3] fit compaction slot, others reserved; reset != 0
 * clears the counters.  Synchronises the device.  The normal build returns QLP_BLS_EUNSUPPORTED (and zeros). */
int qlp_bls_debug_violations(qlp_bls_ctx* ctx, uint64_t* out, int32_t reset);

/* Force the tile class of the fold/scan kernel: 0 = automatic (default); p in 1..9 = no frequency may use a
 * class below p - 1 (class c has 128, 128, 64, 32, 16, 8, 4, 2, 1 columns per CTA for c = 0..8), so that the
 * narrow-column code paths, which real data reach only at very long baselines, are covered on small inputs. */
int qlp_bls_debug_set_path(qlp_bls_ctx* ctx, int32_t path);

#ifdef __cplusplus
}
#endif
#endif /* QLP_BLS_H_ */
