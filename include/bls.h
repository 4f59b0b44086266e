/*
 * bls.h -- C ABI of the B200-native box-least-squares (BLS) periodogram library.
 *
 * What it computes (section 2.2.2): for every light curve of a batch, "phase the
 * light curves at all possible periods and search for a transit-like signal" (L135); at each trial
 * period the curve is phased and "a range of durations and phases" is tested (L145).  The paper
 * names the algorithm (BLS, Kovacs et al. 2002) and prints no formula; the statistic, binning and
 * outputs are the ones BASELINE.json `north_star` fixes and DESIGN.md "Readings" R1-R17 spell out:
 *
 *   per curve      w_i = sigma_i^-2 / sum_j sigma_j^-2 ,  x_i = mag_i - sum_j w_j mag_j
 *   per frequency  fold:  b_i = floor(nb * frac(f * t_i)) ;  W[b] += w_i ;  Y[b] += w_i x_i
 *                  for every start bin a in [0,nb) and width k in [kmin,kmax] (cyclic):
 *                      r = sum_{j<k} W[(a+j) mod nb] ,  s = sum_{j<k} Y[(a+j) mod nb]
 *                      SR(a,k) = s^2 / (r (1-r))        (0 if r(1-r) <= 0)
 *                  report max_{a,k} SR, its (a,k) and depth = s / (r(1-r))  (> 0 = dimming)
 *   per curve      top-k local maxima of the SR spectrum (bls_topk).
 *
 * SR here is the SQUARE of the quantity Kovacs et al. call SR (reading R1); ordering is identical.
 *
 * Conventions
 *   - Every function returns BLS_OK (0) or a negative bls_status.  None throws, aborts or prints.
 *   - "DEVICE" pointers are CUDA device pointers on the plan's device; "HOST" pointers are ordinary
 *     host memory.  The caller owns every batch / output buffer and keeps it alive until the stream
 *     has drained.  The plan owns its copy of the frequency grid and all scratch.
 *   - bls_run / bls_topk only enqueue work on `cuda_stream` (a cudaStream_t passed as void*; NULL =
 *     the legacy default stream).  They synchronise the stream only when plan scratch must grow.
 *   - Structural faults (NULL, bad sizes, CUDA failure) return an error before anything is
 *     launched.  Per-curve DATA faults (fewer than 2 points, non-finite values, sigma <= 0) are
 *     found on the device and reported in status[c]; that curve's spectrum is zero-filled and its
 *     peak list is empty (freq_index = -1), the rest of the batch is unaffected.
 *   - A plan is used by one host thread at a time.  Distinct plans are independent.
 *   - There is no CPU fallback: without a CUDA device bls_plan_create fails with BLS_ERR_CUDA.
 */
#ifndef BLS_B200_H
#define BLS_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    BLS_OK = 0,
    BLS_ERR_NULL = -1,        /* a required pointer is NULL                                        */
    BLS_ERR_CONFIG = -2,      /* bad bls_config (sizes, q range, bin count, frequency grid)        */
    BLS_ERR_BATCH = -3,       /* bad bls_batch (negative count, NULL arrays)                       */
    BLS_ERR_ARG = -4,         /* bad call argument (k out of range, topk before run)               */
    BLS_ERR_CUDA = -5,        /* a CUDA call failed (no device, out of memory, launch failure)     */
    BLS_ERR_UNSUPPORTED = -6, /* shape the kernels cannot hold (curve too long for shared memory)  */
    BLS_ERR_CAPACITY = -7     /* bls_variability_noalloc only: more stars or cells than its fixed,
                                 built-in scratch holds (BLS_NOALLOC_MAX_STARS / _MAX_CELLS)        */
} bls_status;

/* per-curve data status written to bls_outputs.status / readable after bls_run */
#define BLS_CURVE_OK 0
#define BLS_CURVE_TOO_FEW 1      /* fewer than 2 points                    */
#define BLS_CURVE_NONFINITE 2    /* NaN/Inf in t, mag or sigma             */
#define BLS_CURVE_BAD_SIGMA 3    /* some sigma <= 0                        */

typedef struct bls_plan bls_plan; /* opaque */

/* Trial grid and capacities (BASELINE.json north_star: "frequency grid, bin count, duration
 * fraction range").  Copied by bls_plan_create; the caller may free `freqs` afterwards. */
typedef struct {
    int32_t struct_size;   /* = sizeof(bls_config)                                                  */
    int32_t device;        /* CUDA device ordinal                                                   */
    int64_t n_freq;        /* 1 <= nf <= 2^27                                                       */
    const double *freqs;   /* HOST, nf trial frequencies in cycles/day, finite, > 0; NULL = uniform */
    double f0, df;         /* used iff freqs == NULL: f_k = f0 + k*df evaluated in fp64 (R13)       */
    int32_t n_bins;        /* nb >= 4; one bin buffer, (nb + kmax) rows of 256 B plus 5 KB, must fit the
                              227 KB of shared memory a CTA can have: nb + kmax <= 888 (nb <= 807 at
                              q_max = 0.1), else bls_plan_create returns BLS_ERR_UNSUPPORTED              */
    double q_min, q_max;   /* 0 < q_min <= q_max <= 0.5; widths kmin..kmax bins by reading R9:
                              kmin = max(1, floor(q_min*nb + 1e-9)), kmax = min(nb-1, ceil(q_max*nb - 1e-9)) */
    int32_t max_top_k;     /* 1..32: upper bound for bls_topk's k                                   */
    int64_t scratch_bytes; /* budget for the plan-owned spectrum scratch; 0 = default (2 GiB)       */
    uint32_t flags;        /* BLS_FLAG_*                                                            */
} bls_config;

#define BLS_FLAG_NONE 0u
#define BLS_FLAG_CANONICAL_PHASE 1u /* compute every bin index with the slow 3-rounding fp64 rule
                                       (R8) instead of the guarded fast path; results identical   */

/* Ragged CSR batch of light curves (per star a list of HJD times, calibrated
 * magnitudes and errors).  Curve c owns points [offsets[c], offsets[c+1]). */
typedef struct {
    int64_t n_curves;
    const int64_t *offsets;  /* HOST, [n_curves+1], offsets[0] = 0, non-decreasing                 */
    const float *t;          /* DEVICE, days relative to the curve's own origin; need not be sorted */
    const float *mag;        /* DEVICE, magnitudes (larger = fainter)                              */
    const float *sigma;      /* DEVICE, 1-sigma errors, > 0                                        */
    const double *t_origin;  /* HOST, [n_curves] HJD of t = 0 for each curve, or NULL (= 0); only
                                used to report bls_peak.epoch                                      */
} bls_batch;

/* Optional full-spectrum outputs; any pointer may be NULL = "do not write".  All DEVICE,
 * caller-allocated, row-major [n_curves][nf]. */
typedef struct {
    float *sr;             /* per-frequency max over boxes of s^2/(r(1-r))                          */
    uint16_t *best_start;  /* start bin a in [0,nb) of that box                                     */
    uint16_t *best_width;  /* its width k in [kmin,kmax] bins                                       */
    float *depth;          /* signed s/(r(1-r)) of that box; > 0 = dimming in magnitudes (R2)       */
    int32_t *status;       /* [n_curves] BLS_CURVE_*                                                */
} bls_outputs;

/* One peak of a curve's SR spectrum (reading R14: local maximum, ranked by SR descending then
 * index ascending).  freq_index = -1 pads lists shorter than k. */
typedef struct {
    int32_t freq_index;
    float sr;
    float depth;
    uint16_t start_bin;
    uint16_t width_bins;
    double freq;   /* cycles/day                                                                    */
    double epoch;  /* t_origin[c] + ((start_bin + width_bins/2.0)/nb)/freq : mid-box time of the
                      first box after the origin                                                    */
} bls_peak;

/* what to ask bls_plan_query for */
#define BLS_QUERY_KMIN 1
#define BLS_QUERY_KMAX 2
#define BLS_QUERY_NBINS 3
#define BLS_QUERY_NFREQ 4
#define BLS_QUERY_SCRATCH_BYTES 5   /* device bytes currently owned by the plan                    */

/* Validate cfg, copy the grid to the device, derive kmin/kmax (reading R9: outward rounding of
 * [q_min, q_max] to whole bins; "tests a range of durations") and check the shape fits.
 * *out_plan is set only on success.  Errors: BLS_ERR_NULL, BLS_ERR_CONFIG (sizes, q range, non-finite or
 * non-positive frequency), BLS_ERR_UNSUPPORTED (bins do not fit shared memory), BLS_ERR_CUDA (no device,
 * allocation failure: there is no CPU fallback). */
int bls_plan_create(const bls_config *cfg, bls_plan **out_plan);

/* The hot path ("phase the light curves at all possible periods and search for a transit-like
 * signal"; L145: fold at each trial period, "then tests a range of durations and phases"; SURVEY.md section 8
 * rows a0-a5).  For every curve of `batch` and every frequency of the plan: prep (weights, mean removal:
 * readings R4, R5) -> fold into nb phase bins (R6-R8) -> every cyclic box (start, width) scored by
 * SR = s^2/(r(1-r)) (R1, R10, R11), best box per frequency with canonical ties (R12) -> per-curve peak
 * candidates (R14) kept in the plan for bls_topk / bls_refine.  `out` may be NULL (peaks only); its non-NULL
 * arrays receive the full spectra.  Enqueues on cuda_stream; synchronises it only to grow plan scratch.
 * batch->offsets and batch->t_origin are HOST arrays, read before the call returns whether they are pageable
 * or pinned (they are copied into plan-owned staging first; SURVEY 8(b) proposed device pointers; host metadata
 * lets the call validate structure without a device round trip).
 * Errors: BLS_ERR_NULL, BLS_ERR_BATCH (negative count, offsets[0] != 0, decreasing offsets, a curve longer than
 * 2^25 points), BLS_ERR_UNSUPPORTED, BLS_ERR_CUDA; per-curve data faults go to status[], not to the return. */
int bls_run(bls_plan *plan, const bls_batch *batch, const bls_outputs *out, void *cuda_stream);

/* ---- f2: field-shared cadence ------------------------------------------
 * All stars of a pointing are measured on the same exposures ("about 3,000 M-dwarfs in each
 * pointing"; L115: per-epoch zeropoints, 0-2 % of the epochs rejected per field, quality flags per star), so a
 * field is one epoch list and a dense [stars][epochs] matrix of magnitudes and errors.  An entry whose mag or
 * sigma is not finite, or whose sigma <= 0, is an epoch ABSENT for that star (flagged measurement): it simply
 * does not take part; it is not a data fault.  The result for each star is by definition that of bls_run on the
 * star's present epochs.  Where three bin buffers and the field's epochs fit shared memory at least twice per SM
 * (e.g. 64 bins and 140-300 epochs, the paper's cadence; 200 bins do not), the fold computes each epoch's phase
 * and bin index once per (epoch, frequency) for three stars at a time (1.7x the per-star
 * fold as an instruction mix); other shapes run the per-star kernels of bls_run on the field layout. */
typedef struct {
    int64_t n_stars;
    int64_t n_epochs;        /* >= 1                                                                  */
    const float *t;          /* DEVICE [n_epochs] days relative to the field's origin, shared by every star */
    const float *mag;        /* DEVICE [n_stars][n_epochs] row-major                                  */
    const float *sigma;      /* DEVICE [n_stars][n_epochs]                                            */
    const double *t_origin;  /* HOST, ONE value (HJD of t = 0) or NULL                                */
} bls_field_batch;

/* bls_run for a field: same outputs, same bls_topk / bls_refine afterwards (curve index = star index).
 * A star with fewer than 2 present epochs gets status BLS_CURVE_TOO_FEW; a non-finite epoch time makes every
 * star BLS_CURVE_NONFINITE. */
int bls_run_field(bls_plan *plan, const bls_field_batch *field, const bls_outputs *out, void *cuda_stream);

/* a5 Output (the candidates of PAPER.md L151): write the k best peaks of every
 * curve of the last bls_run / bls_run_field to peaks (DEVICE, [n_curves*k]); reading R14 defines a peak
 * (local maximum of the SR spectrum, plateaus to the leftmost sample) and the ranking (SR descending, then
 * index).  1 <= k <= max_top_k, else BLS_ERR_ARG; BLS_ERR_ARG too if nothing has been run.  Enqueues on
 * cuda_stream (the stream of that run, or one ordered after it). */
int bls_topk(bls_plan *plan, int32_t k, bls_peak *peaks, void *cuda_stream);

/* Minimum separation between the peaks of a curve, in steps of the frequency grid (SURVEY.md section 8(c) reading 14;
 * the candidates of PAPER.md L151).  On a fine grid (C3: 500,000 frequencies) the highest local maxima around one
 * signal are its own sidelobes and fill every slot of the list.  With steps > 0 the list is built greedily: peaks
 * (reading R14) are taken in (SR descending, index ascending) order and one is accepted iff its index is MORE than
 * `steps` away from every peak accepted before it; a rejected peak suppresses nothing.  0 (the default) is plain
 * R14.  Takes effect at the next bls_run / bls_run_field / bls_search_host (the peak candidates are picked there);
 * bls_topk and bls_refine then see the separated list.  0 <= steps <= 2^27, else BLS_ERR_ARG. */
int bls_plan_set_peak_min_sep(bls_plan *plan, int32_t steps);

/* Convenience for callers whose data lives in HOST memory: copies the batch to the device, runs
 * bls_run + bls_topk, copies peaks (HOST, [n_curves*k]) and status (HOST, [n_curves], may be NULL)
 * back, and synchronises.  host_batch uses HOST pointers for t / mag / sigma as well. */
int bls_search_host(bls_plan *plan, const bls_batch *host_batch, int32_t k, bls_peak *peaks,
                    int32_t *status);

/* Diagnostic: bins[i] = the phase bin the fold kernel assigns to time t[i] (days) at frequency f[i]
 * (cycles/day) with nb bins -- the same device function the search kernel uses (guarded fast phase,
 * canonical fp64 rule inside the guard band; flags = BLS_FLAG_CANONICAL_PHASE forces the latter).
 * f, t, bins: DEVICE arrays of n entries; *n_canonical (HOST, may be NULL) receives how many pairs
 * took the canonical rule.  Synchronises.  Valid for |f t| < 2^18 cycles. */
int bls_debug_fold_bins(int32_t device, const double *f, const double *t, int64_t n, int32_t n_bins,
                        uint32_t flags, int32_t *bins, int64_t *n_canonical);

/* Diagnostic, the same for the SHIFTED bin grids of bls_refine (reading S3): the grid starts at phase
 * h / (n_shift * n_bins) cycles, 0 <= h < n_shift <= 8, and the fold uses the additive constant and the wider guard
 * band (2 nb + 8 units) it uses inside bls_refine -- also for h = 0.  bins[i] must equal the oracle's
 * oracle_bin_shift(f[i], t[i], n_bins, h / (n_shift * n_bins)).  Arguments and errors as above. */
int bls_debug_fold_bins_shift(int32_t device, const double *f, const double *t, int64_t n, int32_t n_bins, int32_t h,
                              int32_t n_shift, uint32_t flags, int32_t *bins, int64_t *n_canonical);

/* ---- f1: peak significance and refinement ("high-confidence"
 * candidates; readings S1-S4 of DESIGN.md section 3) ------------------------------------------------
 *   S1  sde = (SR_peak - mean(SR)) / sd(SR) over the curve's whole coarse spectrum (population sd);
 *   S2  fine grid of a peak at coarse index q: f_j = f_lo + j*step, j = 0..n_fine-1,
 *       f_lo = freqs[max(q-1,0)], step = (freqs[min(q+1,nf-1)] - f_lo)/(n_fine-1);
 *   S3  the bin grid shifted by s_h = h/(n_shift*nb) cycles, h = 0..n_shift-1: b = floor(nb*frac(f t - s_h));
 *   S4  the refined peak is the best box over (j, h), ties to the smallest j, then h.               */
typedef struct {
    int32_t freq_index;    /* coarse index of the peak this refines; -1 pads short lists            */
    int32_t fine_index;    /* j of the refined frequency (-1: nothing found)                        */
    int32_t shift_index;   /* h of the bin-grid shift                                               */
    uint16_t start_bin;    /* start bin a in the shifted grid                                       */
    uint16_t width_bins;   /* width k                                                               */
    float sr;              /* refined SR                                                            */
    float depth;           /* refined depth (> 0 = dimming)                                         */
    float sde;             /* S1, from the COARSE spectrum and the coarse peak's SR                 */
    float coarse_sr;       /* SR of the coarse peak                                                 */
    double freq;           /* refined frequency, cycles/day                                         */
    double period;         /* 1 / freq, days                                                        */
    double epoch;          /* t_origin[c] + ((a + k/2)/nb + s_h)/freq : mid-box time                */
    double duration;       /* (k/nb)/freq, days                                                     */
} bls_refined_peak;

/* Refine the k best peaks of every curve of the last bls_run: for each, the BLS search of bls_run over
 * its n_fine x n_shift fine entries (2 <= n_fine <= 256 or n_fine == 1; 1 <= n_shift <= 8), reduced to one
 * bls_refined_peak.  out: DEVICE, [n_curves*k].  The batch buffers of that bls_run must still be alive
 * (the plan keeps its prepared copy; t_origin is re-read from the plan's copy).  Enqueues on cuda_stream
 * (the stream of that bls_run or one ordered after it); synchronises only if plan scratch must grow.  */
int bls_refine(bls_plan *plan, int32_t k, int32_t n_fine, int32_t n_shift, bls_refined_peak *out, void *cuda_stream);

/* ---- f3: high-variability pre-filter (section 2.2.1) --------------------------------
 * "We estimate the value and scatter of the locally expected photometric stability as a function of
 * stellar magnitude in 0.1-mag bins, using a sigma-clipped average of the stars detected on each chip.
 * Objects that show a more than 2 sigma increased variability compared to the ensemble expectation are
 * flagged for further review."  Readings V1-V5:
 *   per star   mu = weighted mean magnitude, rms = sqrt(sum_i w_i (mag_i - mu)^2), w as in bls_run;
 *   cell       (group[c], floor((mu - mag_lo)/mag_bin)); stars with a data fault, a group outside
 *              [0, n_groups) or a magnitude outside the n_mag_bins bins belong to no cell (cell = -1);
 *   per cell   sigma clip of the members' rms: E = mean, S = population standard deviation, drop
 *              |rms - E| > clip*S, at most max_iter rounds, stop when nothing is dropped;
 *   flag       1 iff the cell kept >= min_members stars and rms > E + nsig*S.                        */
typedef struct {
    int32_t struct_size;   /* = sizeof(bls_variability_config)                                      */
    int32_t n_groups;      /* >= 1: number of groups (chips)                                        */
    double mag_lo;         /* lower edge of the first magnitude bin                                 */
    double mag_bin;        /* bin width in magnitudes (the paper: 0.1), > 0                         */
    int32_t n_mag_bins;    /* >= 1; n_groups * n_mag_bins <= 2^24                                   */
    int32_t max_iter;      /* clip rounds, 0..100                                                   */
    double clip;           /* clip threshold in sigma (> 0), e.g. 3                                 */
    double nsig;           /* flag threshold in sigma (the paper: 2)                                */
    int32_t min_members;   /* cells that keep fewer stars flag nothing                              */
    int32_t reserved;
} bls_variability_config;

/* All DEVICE, [n_curves] each; any pointer may be NULL = "do not write". */
typedef struct {
    int32_t *status;    /* BLS_CURVE_*                                                               */
    double *mean_mag;   /* mu                                                                        */
    double *rms;        /* weighted RMS about mu                                                     */
    int32_t *cell;      /* group * n_mag_bins + bin, or -1                                           */
    double *expected;   /* E of the star's cell (0 if none)                                          */
    double *scatter;    /* S of the star's cell                                                      */
    int32_t *kept;      /* stars the clip kept in the cell                                           */
    int32_t *flag;      /* 1 = more than nsig sigma above the ensemble expectation                   */
} bls_variability_outputs;

/* Runs the pre-filter on `batch` (same layout as bls_run: offsets HOST, t/mag/sigma DEVICE; t is only
 * checked for finiteness).  group: DEVICE int32 [n_curves] or NULL (= one group).  Enqueues on
 * cuda_stream; scratch is stream-ordered (cudaMallocAsync) and freed before returning control of the
 * stream.  Needs no plan.  Errors: BLS_ERR_NULL / BLS_ERR_CONFIG / BLS_ERR_BATCH / BLS_ERR_CUDA. */
int bls_variability(int32_t device, const bls_variability_config *cfg, const bls_batch *batch,
                    const int32_t *group, const bls_variability_outputs *out, void *cuda_stream);

/* ---- f3 without any allocation ---------------------------------------------------------------------
 * bls_variability needs about 40 bytes of working memory per star (a device copy of the offsets, the cell
 * membership lists of its counting sort, the clip's keep marks) and gets it from cudaMallocAsync.  Some
 * programs that want the pre-filter cannot allocate at the point where they call it:
 *   - a pipeline stage inside a process that has already given all of the GPU's free memory to its own pool
 *     (a tensor framework's caching allocator, a serving runtime): a fresh cudaMalloc there simply fails;
 *   - a per-exposure reduction loop with a latency bound: cudaMalloc / cudaFree may stall the whole device
 *     while they run and may fail half way through a night;
 *   - code that is handed a stream by its host application and is forbidden to create, grow or touch any
 *     memory pool of that application.
 * bls_variability_noalloc is the same filter (same kernels, same order, same results bit for bit) whose
 * working memory is one fixed array compiled into the library, so the call makes no cudaMalloc, cudaMallocAsync,
 * cudaFree or other allocating call.  The price:
 *   - a hard size limit: n_curves <= BLS_NOALLOC_MAX_STARS and n_groups * n_mag_bins <= BLS_NOALLOC_MAX_CELLS
 *     (a PTF pointing has about 3,000 M-dwarfs on 11 chips; 12 chips x 80 bins = 960 cells).
 *     Anything larger returns BLS_ERR_CAPACITY before touching the GPU; use bls_variability for it;
 *   - BLS_NOALLOC_SCRATCH_BYTES (about 0.6 MB) of device memory is held by every GPU on which this library
 *     is loaded, from load until the process exits, whether or not this function is ever called;
 *   - the array is shared by every call on that GPU and still holds what the previous call left there.  The
 *     function itself re-zeroes the one part that has to start at zero (the per-cell member counts) on the
 *     caller's stream and overwrites the rest before reading it, so calls issued one after another on ONE
 *     stream are safe.  Two calls that can run on the GPU at the same time (different streams without an
 *     event between them, two host threads) write over each other's working memory and give wrong results:
 *     the caller serialises them;
 *   - the first call on each GPU looks up where the array lives on that GPU (one cudaGetSymbolAddress, no
 *     allocation) and remembers it.  Make that first call during start-up, before any stream capture is
 *     begun on the device.
 * Inputs and outputs are passed exactly as for bls_variability (outputs left NULL are simply not written;
 * the intermediate ones among them live in the built-in array instead).  batch->offsets (HOST) is copied into
 * the built-in array with cudaMemcpyAsync: if it lives in pinned memory, keep it unchanged until the stream
 * has passed the call.
 * Errors: those of bls_variability, plus BLS_ERR_CAPACITY, plus BLS_ERR_ARG for device outside [0, 64). */
#define BLS_NOALLOC_MAX_STARS 16384
#define BLS_NOALLOC_MAX_CELLS 4096
#define BLS_NOALLOC_SCRATCH_BYTES 655872
int bls_variability_noalloc(int32_t device, const bls_variability_config *cfg, const bls_batch *batch,
                            const int32_t *group, const bls_variability_outputs *out, void *cuda_stream);

/* ---- f4: eclipse detection efficiency of a cadence (Fig. 13; used at L426) ----------
 * "The detection efficiency is the probability that at least two eclipses will be observed from an eclipsing
 * target with a specified period, after observing window and weather effects have been taken into account."
 * Readings W1-W4: the cadence is the epoch list t of each curve of `batch` (only
 * offsets and t are read; t sorted ascending); for each of the n_freq target frequencies (HOST, cycles/day)
 * and each of the n_phase mid-eclipse phases (k + 1/2)/n_phase an epoch is in eclipse iff
 * |x - rint(x)| <= h, x = RN(RN(f t) - phase), h = RN(RN(duration/2) f); the target is detected iff at least
 * min_events distinct eclipses (cycles rint(x)) are observed.
 *   count      DEVICE int32 [n_curves*n_freq] detected phases, or NULL
 *   efficiency DEVICE double [n_curves*n_freq] = count / n_phase, or NULL
 * duration in days (> 0); 1 <= n_phase <= 2^20; min_events >= 1; n_curves <= 65535.  Needs no plan;
 * scratch is stream-ordered.  Enqueues on cuda_stream. */
int bls_detection_efficiency(int32_t device, const bls_batch *batch, int64_t n_freq, const double *freqs,
                             double duration, int32_t n_phase, int32_t min_events, int32_t *count,
                             double *efficiency, void *cuda_stream);

/* ==== UNSTABLE: development switches and launch introspection, for tests, profiling and bench.py ========
 * Nothing below is part of the supported interface: values, meanings and existence may change with the
 * kernels.  A caller that only wants periodograms needs none of it (flags = BLS_FLAG_NONE or
 * BLS_FLAG_CANONICAL_PHASE; queries 1-5). */
#define BLS_FLAG_SINGLE_BUFFER 2u    /* tuning: always use the single-buffer search kernel (every warp
                                       does every phase, full-size CTAs) instead of the warp-specialised,
                                       double-buffered one.                                        */
#define BLS_FLAG_NO_SMALL_CTAS 4u    /* tuning: never use the small-CTA launch shape (kernel 1 with CTAs of two
                                       warps) that small shapes get by default.                     */
#define BLS_FLAG_WARP_PER_TILE 8u    /* tuning: use the one-warp-per-tile search kernel (kernel 3, warp-private
                                       bins) where it fits.                                        */
/* What every kernel-selection flag (SINGLE_BUFFER, NO_SMALL_CTAS, WARP_PER_TILE, WARPS, FOLD_WARPS, WS_SHAPE,
 * MERGE_WARPS) may change: which of several NEAR-TIED boxes of a frequency (fp32 ranking values within 1e-6
 * relative of each other) is reported, because the kernels walk the boxes in different orders before the exact
 * integer merge.  Bin contents, SR of the reported box (computed exactly from its integer sums), statuses and
 * everything else are identical.  CANONICAL_PHASE and FOLD_DEPTH change nothing at all. */
#define BLS_FLAG_WARPS(n) (((uint32_t)(n) & 0xffu) << 8) /* tuning: warps per CTA that walk the boxes
                                       (kernel 1: 1..10, all its warps; kernel 2: 1..19 search warps;
                                       0 = the library's choice).                                  */
#define BLS_FLAG_FOLD_WARPS(n) (((uint32_t)(n) & 0xffu) << 16) /* tuning: warps per CTA that fold, in
                                       the warp-specialised kernel (0 = the library's choice; box +
                                       fold warps <= 20).                                          */

#define BLS_FLAG_WS_SHAPE(n) (((uint32_t)(n) & 7u) << 4) /* tuning: launch shape of the warp-specialised kernel:
                                       1 = 20 warps at equal registers (what WARPS / FOLD_WARPS address; the fold
                                       warps also merge), 2 = 8 search + 4 merge + 16 fold warps, 3 = 12 + 4 + 12,
                                       registers moved from the other roles to the search warps with setmaxnreg
                                       (0 = the library's choice).                                 */
#define BLS_FLAG_MERGE_WARPS(n) (((uint32_t)(n) & 7u) << 24) /* tuning: warps per CTA that share the exact
                                       merge of a tile, 1..7 (0 = the library's choice).           */

#define BLS_FLAG_NO_FIELD_KERNEL (1u << 29) /* tuning: bls_run_field never uses the field kernel (kernel 4: three stars
                                       per CTA share each epoch's bin index) and runs the per-star kernels of bls_run.
                                       Like the other kernel-selection flags: near-tied boxes only.          */

#define BLS_FLAG_FOLD_DEPTH(n) (((uint32_t)(n) & 3u) << 27) /* tuning: groups of 4 points a fold warp keeps in
                                       flight, 1 or 2 (0 = the library's choice).  Never changes results. */

#define BLS_QUERY_LAST_LAUNCHES 6   /* kernels launched by the last bls_run + bls_topk            */
#define BLS_QUERY_LAST_CANONICAL 7  /* point-folds of the last bls_run that took the canonical
                                       fp64 bin rule because the fast phase fell in its guard band
                                       (synchronises the stream of that run)                       */
#define BLS_QUERY_TILE_FREQS 8      /* frequencies per CTA work item in the search kernel          */
#define BLS_QUERY_SEARCH_CTAS 9     /* CTAs of the last search launch                              */
#define BLS_QUERY_LAST_SEARCH_NS 10 /* device time (ns, CUDA events on the run's stream) the search
                                       kernel launches of the last bls_run took (synchronises)    */
#define BLS_QUERY_SEARCH_KERNEL 11  /* search kernel of the last run: 1 = single buffer (all warps do every
                                       phase; also the small-CTA shape of small configurations),
                                       2 = warp-specialised double buffer, 3 = one warp per tile,
                                       4 = field kernel of bls_run_field (0 = none yet)            */
#define BLS_QUERY_LAST_SEARCH_LAUNCHES 12 /* search kernel launches of the last bls_run (one per chunk of
                                       curves): LAST_SEARCH_NS / this = the average launch duration */
#define BLS_QUERY_WS_SHAPE 13       /* launch shape of the warp-specialised kernel in the last run: 0 = equal registers,
                                       the fold warps merge; 1 = 8 search + 4 merge + 16 fold warps; 2 = 12 + 4 + 12
                                       (-1 = another kernel ran)                                  */
/* ==== end of the unstable block ==================================================================== */

/* NULL is a no-op. */
int bls_plan_destroy(bls_plan *plan);

/* Derived constants and counters of the plan (BLS_QUERY_*): kmin / kmax of reading R9, so callers never
 * re-derive them; launch facts of the last run.  BLS_ERR_ARG for an unknown `what` or a last-run query before
 * any run.  Queries 7 and 10 synchronise the stream of the last run. */
int bls_plan_query(const bls_plan *plan, int32_t what, int64_t *value);

/* Static string for a bls_status (never NULL). */
const char *bls_strerror(int status);

/* Last CUDA error string seen by this plan (static storage owned by the plan; "" if none). */
const char *bls_plan_last_cuda_error(const bls_plan *plan);

#ifdef __cplusplus
}
#endif
#endif /* BLS_B200_H */
