/*
 * gpfc.h -- C ABI of libgpfc.so: B200-native GPU phase folding + noise
 * normalisation, the data-parallel hot path of GPFC (arXiv 2312.02063,
 * "PAPER.md" below; line numbers refer to /root/reference/PAPER.md).
 *
 * What the path computes (one "fold" per (light curve, trial period) pair):
 *   step 1  u = t - t0, x = u / P, phi = x - floor(x)      PAPER.md:87(1), :111 "First"
 *   step 2  k = min(trunc(phi * nbins), nbins - 1)          PAPER.md:105, :111 "Secondly"
 *   step 3  sum[k] += flux, count[k] += 1                   PAPER.md:111 "Thirdly"
 *   step 5  mean[k] = sum[k] / count[k]                     PAPER.md:111 "Lastly"
 *   normalise: out[k] = mu + (mean[k] - mu) / s, mu and s the mean and the
 *           population standard deviation of mean[] over the non-empty bins;
 *           empty bins get mu
 * The phase formula is exactly the one above in IEEE fp64 with no FMA
 * contraction (true division); the kernels use a reciprocal multiply with a
 * guard band and fall back to the division wherever the two could differ, so
 * bin indices are bit-identical to that formula.
 *
 * Conventions for every call
 *   - Pointers marked "device" must be device-accessible memory of the
 *     current CUDA device; pointers marked "host" are ordinary host memory.
 *     All memory is owned by the caller.  Nothing is retained after the work
 *     is enqueued, except the workspace registered with gpfc_set_workspace.
 *   - Device-pointer calls are asynchronous on the calling thread's current
 *     gpfc stream (gpfc_set_stream; default: the legacy default stream) and
 *     never synchronise the host or any stream; they can be captured in a CUDA
 *     graph (register a workspace first: gpfc_set_workspace).  *_host calls
 *     are synchronous.
 *   - One process may drive several devices: the library keeps its per-device
 *     state (kernel attributes, SM count) keyed by cudaGetDevice() and sets it
 *     up on the first call made with that device current, or in gpfc_init().
 *     Pointers, stream and workspace must belong to the current device.
 *   - Alignment: times 8 bytes, everything else 4 bytes.  Outputs that are
 *     16-byte aligned (any torch allocation) are written with vector stores;
 *     other alignments are accepted and take scalar stores.
 *   - Return value: a gpfc_status (0 = success).  On failure
 *     gpfc_last_error() describes it; outputs are then unspecified.
 *   - Sizes of 0 (n, nperiods, ncurves, nprofiles) are valid no-ops.
 *   - nbins: 1 <= nbins <= GPFC_MAX_NBINS.  Any value is accepted; every
 *     nbins <= 256 and the powers of two up to 4096 take the fast kernels, other
 *     values a plain one (true division per point-period, ~100x slower, counted
 *     by gpfc_path_counters).
 *   - Outputs are fully overwritten, layout row-major [curve][period][bin].
 *   - Data conventions (cannot be checked on the host): a sample whose time
 *     or flux is not finite is skipped (not counted); a period that is not
 *     finite and positive yields an all-zero row (sum, count and norm).
 *   - Sums are accumulated exactly in per-curve fixed point (DESIGN.md
 *     "Accumulation"): for flux that is a multiple of 2^-s on the curve's
 *     scale the sums are exact and independent of order.
 *   - There is no CPU fallback: without a CUDA device every compute call
 *     returns GPFC_ERR_CUDA.
 */
#ifndef GPFC_H
#define GPFC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    GPFC_OK = 0,
    GPFC_ERR_INVALID_ARG = 1,  /* NULL required pointer, negative size, bad range  */
    GPFC_ERR_UNSUPPORTED = 2,  /* nbins out of range                               */
    GPFC_ERR_WORKSPACE = 3,    /* registered workspace too small / allocation failed */
    GPFC_ERR_CUDA = 4,         /* CUDA runtime error (text in gpfc_last_error)     */
    GPFC_ERR_ABORTED = 5       /* a caller-supplied callback returned non-zero     */
} gpfc_status;

#define GPFC_MAX_NBINS 4096
/* limits of gpfc_fold_noalloc (its scratch is a static device array sized for them) */
#define GPFC_NOALLOC_MAX_SAMPLES 131072
#define GPFC_NOALLOC_MAX_PERIODS 262144

/* gpfc_make_period_grid mode_flags: spacing | endpoint */
enum { GPFC_GRID_UNIFORM_FREQUENCY = 0, GPFC_GRID_UNIFORM_PERIOD = 1 };
enum { GPFC_GRID_ENDPOINT_INCLUSIVE = 0, GPFC_GRID_ENDPOINT_EXCLUSIVE = 2 };

/* Library version string (static storage). */
const char *gpfc_version(void);

/*
 * Optional: set up the library's per-device state for the CURRENT device now
 * (opt-in shared-memory attributes of the kernels, SM count).  Every compute
 * call does the same on its first use of a device; nothing in it touches a
 * stream, so calling it is never required, not even before graph capture.
 */
int gpfc_init(void);

/* Text of the calling thread's last error (static thread-local storage; never NULL). */
const char *gpfc_last_error(void);

/* Set the calling thread's stream (a cudaStream_t passed as void*; NULL = legacy
 * default stream).  Every later device-pointer call of this thread is enqueued on it. */
int gpfc_set_stream(void *cuda_stream);

/*
 * Scratch memory.  The fold needs, per call, room for the pre-processed
 * samples (u = t - t0 in fp64, fixed-point flux), per-curve and per-period
 * tables: gpfc_workspace_bytes() returns an upper bound for a call of the given
 * size.  If a workspace registered with gpfc_set_workspace() (device memory,
 * 256-byte aligned, owned by the caller, must stay valid until the work that
 * uses it has finished) is large enough it is used; otherwise the library
 * allocates and frees scratch stream-ordered (cudaMallocAsync) inside the call.
 * gpfc_set_workspace(NULL, 0) unregisters.  Per-thread, like the stream.
 * With nbins >= 512 and more than 65,408 samples in the call the bound includes
 * a 32-bit count overflow area (128 KB per SM, see fold_pk.cu).
 */
size_t gpfc_workspace_bytes(int64_t ncurves, int64_t n_total, int64_t nperiods, int nbins);
int gpfc_set_workspace(void *dev_ptr, size_t bytes);

/*
 * Trial-period grid (Eq. 1 and "uniformly sample 100,000
 * periods within [0.2, 1.0] days").  D = nperiods - 1 (inclusive) or nperiods
 * (exclusive), at least 1.
 *   frequency mode: f_j = 1/pmax + ((1/pmin - 1/pmax) * j) / D, periods_out[j] = 1 / f_j
 *                   (ascending frequency, i.e. descending period)
 *   period mode:    periods_out[j] = pmin + ((pmax - pmin) * j) / D
 * every operation individually rounded to fp64 (no FMA).
 * periods_out: device, fp64 [nperiods].  pmin <= 0, pmax < pmin, non-finite
 * bounds or nperiods < 0 -> GPFC_ERR_INVALID_ARG.
 */
int gpfc_make_period_grid(double pmin, double pmax, int64_t nperiods, int mode_flags,
                          double *periods_out);

/* Eq. 1: N_sample = N_o * T / L.  Host-only helper for sizing the grid. */
double gpfc_n_sample(double n_o, double t_window, double l_width);

/*
 * Fold one light curve over a set of trial periods (steps 1-3: PAPER.md:87(1), :111
 * "First" to "Thirdly").
 *   times    device fp64 [n]     sample times (irregular allowed: PAPER.md:334; any order is
 *                                accepted and gives the same result, but only time-ordered
 *                                input is fast: the kernels handle samples in tiles of 128
 *                                consecutive samples whose time span must stay well below
 *                                2^20 / nbins periods, other tiles take the exact division
 *                                for every point-period, ~10x slower; gpfc_path_counters
 *                                reports how many work items did)
 *   flux     device fp32 [n]     detrended, median-subtracted relative flux
 *   periods  device fp64 [nperiods]
 *   t0       reference epoch subtracted from every time first
 *   out_sum  device fp32 [nperiods][nbins]   per-bin flux sums   (may be NULL)
 *   out_count device u32 [nperiods][nbins]   per-bin counts      (may be NULL)
 */
int gpfc_fold(const double *times, const float *flux, int64_t n,
              const double *periods, int64_t nperiods, int nbins, double t0,
              float *out_sum, uint32_t *out_count);

/*
 * gpfc_fold plus the fused noise normalisation (PAPER.md:111 "First" to "Lastly", :63), for
 * callers that must not allocate: code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc.  This call allocates NOTHING, with or without gpfc_set_workspace: no
 * cudaMalloc / cudaMallocAsync / cudaFree, no event creation (gpfc_profile does not time it).
 * Its scratch (valid samples as fixed-point records, per-period reciprocals) is a static device
 * array inside the library: 4.8 MB that every GPU which loads the library holds until exit.
 * Arguments as gpfc_fold; out_norm device fp32 [nperiods][nbins] (may be NULL) as out_norm of
 * gpfc_fold_batch.  Asynchronous on the thread's stream like every device-pointer call.
 * Limits (GPFC_ERR_UNSUPPORTED with a message beyond them, nothing is launched):
 *   n <= GPFC_NOALLOC_MAX_SAMPLES (131072), nperiods <= GPFC_NOALLOC_MAX_PERIODS (262144), and
 *   n <= 65408 when nbins is 512, 1024, 2048 or 4096 (longer curves need the count overflow
 *   area of that kernel, which is not part of the static scratch).
 * All calls, from every host thread and stream, share the one array of their device: two calls
 * whose kernels overlap on the GPU race (wrong results, no error).  Issue them on one stream, or
 * order them with events.  The array keeps the previous call's contents; nothing in it has to
 * start at zero (the prepass rewrites every word the fold reads), so nothing is cleared.
 */
int gpfc_fold_noalloc(const double *times, const float *flux, int64_t n,
                      const double *periods, int64_t nperiods, int nbins, double t0,
                      float *out_sum, uint32_t *out_count, float *out_norm);

/*
 * Step 5 + noise normalisation of nprofiles folded profiles (PAPER.md:111
 * "Lastly", :63).  sum, count: device [nprofiles][nbins]; out_norm: device fp32
 * [nprofiles][nbins].  All-empty profile -> zeros; fewer than two non-empty
 * bins or zero spread -> mu everywhere.  Arithmetic in fp64.
 */
int gpfc_normalize(const float *sum, const uint32_t *count, int64_t nprofiles, int nbins,
                   float *out_norm);

/*
 * NEXT row: step 4 of the paper's fold, "Fourthly",
 * Fig. 4(c): merge the nb1 equal-width intermediary bins of each folded profile (e.g. 4096,
 * from gpfc_fold) into nb2 final bins (e.g. 256) that each contain the same number of points,
 * scanning left to right and splitting a boundary bin pro rata by count (R18).
 *   sum, count   device [nprofiles][nb1]   (outputs of gpfc_fold / gpfc_fold_batch)
 *   out_mean     device fp32 [nprofiles][nb2]  mean flux of each final bin   (may be NULL)
 *   out_norm     device fp32 [nprofiles][nb2]  the same profile noise-normalised as in
 *                gpfc_normalize (every final bin counts as non-empty)        (may be NULL)
 * A profile without points gives zeros.  Arithmetic in fp64; the input sums are fp32, so the
 * merged means carry their rounding (6e-8 relative to the flux level: for a normalised profile
 * of an UNCENTRED relative flux near 1 with a spread of a few 1e-4 that is ~1e-4 of its unit;
 * median-subtracted flux, as gpfc_fold asks for, or gpfc_fold_two_tier do not have this limit).
 */
int gpfc_merge_equal_count(const float *sum, const uint32_t *count, int64_t nprofiles, int nb1,
                           int nb2, float *out_mean, float *out_norm);

/*
 * Batched fold, optionally fused with the normalisation: steps 1-3 and 5 of PAPER.md:111
 * ("First", "Secondly", "Thirdly", "Lastly") for every (curve, trial period) pair -- the
 * paper folds one curve at 100,000 periods, 16 at a time (:113-115); here a call folds any
 * number of curves over a shared grid -- and the noise normalisation of PAPER.md:63.
 *   times, flux  device, curves stored back to back: curve c is samples
 *                offsets[c] .. offsets[c+1]-1
 *   offsets      device int64 [ncurves + 1], non-decreasing, offsets[0] >= 0
 *   n_total      number of elements in times / flux (>= offsets[ncurves]);
 *                sizes the scratch, read on the host
 *   periods      device fp64 [nperiods], shared by all curves
 *   t0           device fp64 [ncurves], or NULL for 0.0
 *   out_sum, out_count, out_norm   device [ncurves][nperiods][nbins]; any may
 *                be NULL.  out_norm alone is the fused fold + normalise path:
 *                sums and counts never leave shared memory.  out_norm is
 *                computed from the exact sums, not from their fp32 roundings.
 */
int gpfc_fold_batch(const double *times, const float *flux, const int64_t *offsets,
                    int64_t ncurves, int64_t n_total, const double *periods,
                    int64_t nperiods, int nbins, const double *t0,
                    float *out_sum, uint32_t *out_count, float *out_norm);

/*
 * The paper's complete fold, steps 1-5 (Fig. 4): fold at nb1 equal-width
 * intermediary bins (4096 in the paper), merge them left to right into nb2 bins (256) that
 * each hold the same number of points, splitting a bin on a boundary pro rata by count
 * (R18), take the mean of every final bin, and noise-normalise the profile (:63).
 * Arguments as gpfc_fold_batch (offsets may be NULL when ncurves == 1: the curve is then
 * times[0 .. n_total)).
 *   out_mean  device fp32 [ncurves][nperiods][nb2]  mean flux of the final bins   (may be NULL)
 *   out_norm  device fp32 [ncurves][nperiods][nb2]  the same, scaled to population
 *             standard deviation 1 about its mean (every final bin counts)       (may be NULL)
 * For nb1 in {1024, 2048, 4096} and nb2 <= nb1 / 16 (256 for nb1 = 4096, the paper's pair)
 * fold and merge are ONE kernel: the intermediary profile stays in shared memory and the merge
 * reads the exact integer sums.  Any other (nb1, nb2) folds into a temporary intermediary
 * profile (stream-ordered allocation, <= 256 MB; fp32 sums taken relative to the curve's
 * internal center, which the merge adds back) and runs the kernel of gpfc_merge_equal_count.
 * A period that is not finite-positive, or a curve without valid samples, gives zeros.
 */
int gpfc_fold_two_tier(const double *times, const float *flux, const int64_t *offsets,
                       int64_t ncurves, int64_t n_total, const double *periods,
                       int64_t nperiods, int nb1, int nb2, const double *t0,
                       float *out_mean, float *out_norm);

/*
 * Synthetic light curves on the device (PAPER.md 2.6 "Light Curve
 * Simulation": Eq. 2 :162, parameter ranges :166-170, Table 2 :176-180, trapezoid :170,
 * Fig. 7 :188, SNR range :190): white Gaussian noise of per-point standard deviation sigma
 * around 1, with a periodic trapezoidal transit whose depth follows from a requested
 * signal-to-noise ratio through Eq. 2.  The inputs of large sweeps never touch the host.
 *
 * Generator specification (a pure function of seed, curve index c and sample index i, so the
 * CPU oracle reproduces it bit for bit).  Random words come from Philox4x32-10 (Salmon et al.,
 * SC'11) with key (seed low word, seed high word) and counter (w0, w1, w2, w3); U(x) =
 * (x + 1/2) 2^-32; every fp64 operation is rounded once, in the order written, no FMA.
 *   curve c:  (x0..x3) = philox(0, 0, c, 0):  sigma = sigma_lo + (sigma_hi - sigma_lo) U(x0),
 *             r = U(x1), e = U(x2), alpha = snr_lo + (snr_hi - snr_lo) U(x3)
 *             philox(0, 1, c, 0):  the curve carries a transit iff U(x0) < transit_fraction
 *             philox(k, 2, c, 0), k = 0, 1, ... 63:  p = period_lo + (period_hi - period_lo) U(x0),
 *             L = (ratio_lo + (ratio_hi - ratio_lo) U(x1)) p; the first k with
 *             duration_lo <= L <= duration_hi is taken (k = 63: L is clamped) -- Table 2 gives
 *             ranges for p, L and L/p but no joint law (R21)
 *             depth d = (alpha sigma) / sqrt(((double)n L) / p)                 Eq. 2 solved for d
 *             long base T14 = (2 L) / (1 + r), short base T23 = r T14 (duration L at half
 *             depth), mid-transit epoch tc = e p
 *   sample i: t = t_start + (double)i cadence
 *             (x0..x3) = philox(i, 0, c, 1): u1 = ((x0 2^20 + (x1 >> 12)) + 1/2) 2^-52,
 *             u2 = U(x2), z = sqrt(-2 ln u1) cos(2 pi u2)                       (Box-Muller)
 *             ln u:  u = m 2^e with m in [1/2, 1) from the bits of u; if m < 0.70710678118654752
 *                    then m = 2 m, e = e - 1;  s = (m - 1)/(m + 1), w = s s,
 *                    P = 1/23; P = P w + 1/(2j+1) for j = 10 ... 0;
 *                    ln u = e * 0.69314718055994531 + 2 (s P)
 *             cos(2 pi v):  8 v = k + f (k = floor, octant), g = 1 - f if k is odd else f,
 *                    theta = g * 0.78539816339744831, w = theta theta; for k in {1, 2, 5, 6}
 *                    value = theta (1 - w/3! + w^2/5! - ... - w^7/15!), else
 *                    value = 1 - w/2! + w^2/4! - ... + w^8/16! (Horner from the highest term,
 *                    each coefficient the fp64 quotient 1/j!); negated for k in {2, 3, 4, 5}
 *             y = (t - tc) / p; y = y - floor(y + 1/2); x = |y| p
 *             shape = 1 if x <= T23/2, 0 if x >= T14/2, else (T14/2 - x) / (T14/2 - T23/2)
 *             flux = (float)((1 + sigma z) - d shape), minus 1.0f (in fp32) if GPFC_LC_CENTERED
 *
 *   prm       host; ranges as above, gpfc_lc_params_default() fills Table 2's
 *   times     device fp64 [ncurves][n], may be NULL (every curve has the same time stamps)
 *   flux      device fp32 [ncurves][n]
 *   offsets   device int64 [ncurves + 1] = c n, may be NULL (the array gpfc_fold_batch wants)
 *   params_out device fp64 [ncurves][8], may be NULL: {p, L, sigma, d (0 without a transit), r,
 *             tc, alpha, 1.0 or 0.0 = carries a transit}; scratch is taken from the workspace
 *             (8 * 8 * ncurves bytes) or allocated stream-ordered when it is NULL
 * ncurves and n must be below 2^32.  GPFC_ERR_INVALID_ARG for an empty or reversed range.
 */
enum { GPFC_LC_CENTERED = 1, GPFC_LC_NO_NOISE = 2 };
typedef struct {
    double period_lo, period_hi;       /* p,     Table 2: (0.3, 1.0) d            */
    double duration_lo, duration_hi;   /* L,     Table 2: (0.03, 0.09) d          */
    double ratio_lo, ratio_hi;         /* L / p, Table 2: (0.04, 0.12)            */
    double sigma_lo, sigma_hi;         /* sigma, Table 2: (0.0001, 0.0005)        */
    double snr_lo, snr_hi;             /* alpha: [6, 10]            */
    double transit_fraction;           /* share of the curves that carry a transit */
    double cadence, t_start;           /* t_i = t_start + i cadence               */
    int32_t flags;                     /* GPFC_LC_*                               */
    int32_t reserved;
} gpfc_lc_params;
int gpfc_lc_params_default(gpfc_lc_params *prm);
int gpfc_make_light_curves(uint64_t seed, int64_t ncurves, int64_t n, const gpfc_lc_params *prm,
                           double *times, float *flux, int64_t *offsets, double *params_out);

/*
 * Streaming fold for a downstream consumer ("transfer data in
 * batches", :278 the fold of light curve k+1 runs while the CNN scores light curve k): the
 * batch is folded chunk by chunk into one of two device slabs, and every finished chunk is
 * handed to the caller's consumer, which works on it on ITS stream while the next chunk folds.
 *
 * Arguments as gpfc_fold_batch (all device pointers), then
 *   outputs          GPFC_OUT_SUM | GPFC_OUT_COUNT | GPFC_OUT_NORM: the arrays to produce.
 *                    GPFC_OUT_NORM alone is the scorer's input and a third of the bytes.
 *   slab_bytes       bytes of output per chunk (all requested arrays together); 0 = 512 MB
 *                    per requested array.
 *                    A chunk is a run of whole curves; if the profiles of one curve exceed the
 *                    slab, a run of consecutive periods of one curve.
 *   consumer_stream  the stream (cudaStream_t) the consumer's work runs on; NULL = the fold
 *                    stream (no overlap)
 *   on_chunk         called on the calling host thread once per chunk, in order, right after
 *                    the chunk's fold has been ENQUEUED: consumer_stream already waits for
 *                    chunk->ready, so the callback only enqueues its work on that stream
 *                    (kernels, copies) and returns 0 without blocking.  The chunk's arrays are
 *                    device pointers [ncurves][nperiods][nbins] into the slab (NULL for arrays
 *                    not requested), valid for work enqueued on consumer_stream inside the
 *                    callback: the slab is folded into again once that work has run.  A
 *                    non-zero return stops the loop: GPFC_ERR_ABORTED.  The callback must not
 *                    call the fold entry points of this library (the call in progress owns the
 *                    thread's stream and scratch).
 * The library allocates the two slabs stream-ordered on the fold stream and frees them after
 * the consumer stream's last chunk; the host never waits.  Returns when everything is
 * enqueued.
 */
enum { GPFC_OUT_SUM = 1, GPFC_OUT_COUNT = 2, GPFC_OUT_NORM = 4 };
typedef struct {
    int64_t curve0, ncurves;     /* curves   [curve0, curve0 + ncurves)   of the batch */
    int64_t period0, nperiods;   /* periods  [period0, period0 + nperiods) of the grid  */
    int32_t nbins;
    int32_t slot;                /* which of the two slabs (0 / 1)                      */
    const float *sum;            /* device [ncurves][nperiods][nbins] or NULL           */
    const uint32_t *count;
    const float *norm;
    void *ready;                 /* cudaEvent_t recorded on the fold stream after this chunk */
} gpfc_chunk;
typedef int (*gpfc_chunk_fn)(const gpfc_chunk *chunk, void *consumer_stream, void *user);
int gpfc_fold_stream(const double *times, const float *flux, const int64_t *offsets,
                     int64_t ncurves, int64_t n_total, const double *periods, int64_t nperiods,
                     int nbins, const double *t0, int outputs, size_t slab_bytes,
                     void *consumer_stream, gpfc_chunk_fn on_chunk, void *user);

/*
 * Host-buffer convenience entry points (the end-to-end path): same
 * arguments, but every pointer is HOST memory (pinned memory makes the copies
 * faster but is not required).  The call allocates device buffers, copies the
 * inputs in, runs gpfc_fold_stream on the current stream with a consumer that
 * copies every finished chunk back on a second stream (so the copy of chunk k
 * overlaps the fold of chunk k+1), and synchronises both streams before
 * returning.  Pass only out_norm (out_sum, out_count NULL) to move a third of
 * the bytes.
 */
int gpfc_make_period_grid_host(double pmin, double pmax, int64_t nperiods, int mode_flags,
                               double *periods_out);
int gpfc_fold_batch_host(const double *times, const float *flux, const int64_t *offsets,
                         int64_t ncurves, int64_t n_total, const double *periods,
                         int64_t nperiods, int nbins, const double *t0,
                         float *out_sum, uint32_t *out_count, float *out_norm);

/*
 * Measurement hooks for bench.py (per calling thread).  gpfc_profile(1) clears the
 * counters and makes every later fold call record a CUDA-event pair around its
 * fold-kernel launch on the call's stream; gpfc_profile(0) clears and stops.
 * gpfc_profile_read waits for the recorded events and returns the summed
 * fold-kernel time (ms), the number of fold-kernel launches timed, and the number
 * of kernels of this library launched since gpfc_profile() (any may be NULL).
 */
int gpfc_profile(int enable);
int gpfc_profile_read(double *fold_kernel_ms, int64_t *fold_launches, int64_t *kernel_launches);

/*
 * Which slow paths ran since the last gpfc_profile() call (out: host int64[8]):
 *   [0] fold calls of this thread that used the generic kernel (nbins above 256 that is
 *       not a power of two: one CTA per (curve, period), true division for every point-period)
 *   [1] work items (curve x group of periods) of this DEVICE that took the exact division for
 *       every point-period: unsorted times, tiles spanning huge gaps, periods far below the
 *       sampling interval
 *   [2] guard-band re-checks (lane x tile) of this device: normal, ~1e-4 of the tiles
 *   [3] gpfc_fold_two_tier calls of this thread that could not fuse fold and merge
 *   [4] work items of this device (nbins >= 512, curves of more than 65,408 samples) folded
 *       twice because more than 65,535 points of a period fell into one pair of rows: the
 *       second pass flushes the packed 16-bit counts to a 32-bit side array
 *   [5..7] reserved (0)
 * Synchronises the calling thread's stream.
 */
int gpfc_path_counters(int64_t *out);

/*
 * Roofline calibration: runs the library's micro-kernels on
 * the current stream and reports the measured peak rates of the units that
 * bound the fold, so that bench.py can quote its denominator from the same run
 * and clocks.  out (host, double[8]):
 *   [0] conflict-free shared-memory atomic lane-updates / s (ATOMS.ADD + ATOMS.POPC.INC mix)
 *   [1] fp64 (DMUL + DADD) pairs / s
 *   [2] point-periods / s of the fold kernel's inner loop alone (no global loads, tile set-up,
 *       epilogue or barriers): the ceiling of the kernel design
 *   [3] fp32 atomicAdd lane-updates / s on shared memory (a CAS loop on sm_100a), pattern of [0]
 *   [4] plain LDS + add + STS lane-updates / s on warp-private rows (no atomics)
 *   [5..7] reserved (0)
 * Synchronous.
 */
int gpfc_measure_peaks(double *out);

#ifdef __cplusplus
}
#endif
#endif /* GPFC_H */
