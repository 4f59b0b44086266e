/*
 * bls_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the hot path computes: the box-least-squares (BLS)
 * search of PAPER.md section 2.2.2 (L133-147): "phase the light curves at all possible periods and
 * search for a transit-like signal" (L135); per trial period the curve is phased and "a range of
 * durations and phases" is tested (L145).  The paper prints no formula; the statistic is the one
 * BASELINE.json `north_star` fixes, SR = s^2/(r(1-r)), depth = s/(r(1-r)), which is the weighted
 * least-squares fit of a two-level (in-box / out-of-box) signal (derivation: DESIGN.md "The
 * statistic"; checked by brute force in tests/test_oracle_pins.py).  Steps O1..O5 are SURVEY.md
 * section 8(c) / DESIGN.md "Readings".
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or constant with the CUDA
 * library under paper_1112_1701_b200/csrc/ and is never linked into it.
 *
 * Written so it can be checked against the definition by eye: no blocking, no prefix-sum tricks,
 * no SIMD, no reordering.  Every box is summed directly (running sum over its bins, in bin order).
 * Build: gcc -O2 -ffp-contract=off -shared -fPIC (no FMA contraction: the phase rule O4 is a
 * sequence of individually rounded IEEE operations).
 *
 * Pins (tests/test_oracle_pins.py, tests/test_oracle_peaks.py):
 *   oracle_prepare      - weighted-mean identities, weight-scaling invariance          (pinned)
 *   oracle_widths       - table of DESIGN.md reading R9                               (pinned)
 *   oracle_bin          - exact rational arithmetic (fractions.Fraction) + edge cases (pinned)
 *   oracle_spectrum     - brute force over boxes from the least-squares definition,
 *                         brute force over all point subsets (N<=12), noiseless injected box
 *                         with closed-form depth and SR, invariants                   (pinned)
 *   oracle_sr_at        - same brute force, box/complement symmetry                   (pinned)
 *   oracle_peaks        - hand-written spectra with answers written out               (pinned)
 *   oracle_peaks_sep    - hand-written spectra with answers written out (a rejected peak
 *                         suppresses nothing; "more than" is strict), min_sep = 0 equals
 *                         oracle_peaks, brute force over all subsets on small spectra  (pinned)
 *   oracle_sde          - hand-written spectra, closed form                           (pinned)
 *   oracle_bin_shift    - exact rational arithmetic with a bin-grid shift              (pinned)
 *   oracle_detection_efficiency - closed forms on regular cadences (d/P, 2d/P), degenerate cases,
 *                         an event-centred brute force, the integer-day dips of Fig. 13   (pinned)
 *   oracle_refine       - noiseless box between coarse grid points recovered to the fine
 *                         step and to the quarter-bin shift (closed-form SR and depth),
 *                         brute force over boxes with shifted member sets             (pinned)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

/* O1 + O2 (reading R4, R5): w_i = sigma_i^-2 / sum_j sigma_j^-2 ; mu = sum w_i m_i ; x_i = m_i - mu.
 * Sums run in index order.  Returns 0, or a per-curve data fault:
 *   1 = fewer than 2 points, 2 = non-finite t/mag/sigma, 3 = sigma <= 0. */
int oracle_prepare(int64_t n, const float *t, const float *mag, const float *sigma,
                   double *w, double *x)
{
    if (n < 2) return 1;
    for (int64_t i = 0; i < n; ++i) {
        if (!isfinite((double)t[i]) || !isfinite((double)mag[i]) || !isfinite((double)sigma[i]))
            return 2;
        if (!(sigma[i] > 0.0f)) return 3;
    }
    double sw = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        double s = (double)sigma[i];
        sw += 1.0 / (s * s);
    }
    if (!isfinite(sw) || !(sw > 0.0)) return 2;
    double mu = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        double s = (double)sigma[i];
        w[i] = (1.0 / (s * s)) / sw;
        mu += w[i] * (double)mag[i];
    }
    for (int64_t i = 0; i < n; ++i) x[i] = (double)mag[i] - mu;
    return 0;
}

/* O3 (reading R9): trial widths in whole bins, rounded outward from [q_min, q_max]:
 *   kmin = max(1, floor(q_min*nb + 1e-9)),  kmax = min(nb-1, ceil(q_max*nb - 1e-9)). */
void oracle_widths(int nb, double q_min, double q_max, int *kmin, int *kmax)
{
    int lo = (int)floor(q_min * (double)nb + 1e-9);
    int hi = (int)ceil(q_max * (double)nb - 1e-9);
    if (lo < 1) lo = 1;
    if (hi > nb - 1) hi = nb - 1;
    if (hi < lo) hi = lo;
    *kmin = lo;
    *kmax = hi;
}

/* O4 phase rule (reading R8): three individually rounded fp64 operations, no fused multiply-add.
 *   p = RN(f*t) ; phi = p - floor(p) (exact) ; b = trunc(RN(phi*nb)) ; b = nb-1 if b >= nb. */
int oracle_bin(double f, double t, int nb)
{
    volatile double p = f * t;              /* volatile: one rounding, never contracted */
    double phi = p - floor(p);
    volatile double xb = phi * (double)nb;
    int b = (int)xb;
    if (b >= nb) b = nb - 1;
    return b;
}

/* O4 fold ("phases the light curve at that period", L145): W[b] += w_i, Y[b] += w_i x_i. */
static void fold(int64_t n, const float *t, const double *w, const double *x, double f, int nb,
                 double *W, double *Y)
{
    for (int b = 0; b < nb; ++b) { W[b] = 0.0; Y[b] = 0.0; }
    for (int64_t i = 0; i < n; ++i) {
        int b = oracle_bin(f, (double)t[i], nb);
        W[b] += w[i];
        Y[b] += w[i] * x[i];
    }
}

/* O4 box search ("tests a range of durations and phases", L145).  Every start bin a in [0,nb) and
 * every width k in [kmin,kmax]; bins are cyclic (reading R11); each box is a direct running sum in
 * bin order; a box is valid iff r(1-r) > 0 (R10); ties go to the smallest k, then the smallest a
 * (R12).  An all-invalid frequency reports SR = 0, a = 0, k = kmin, depth = 0. */
static void search(int nb, int kmin, int kmax, const double *W, const double *Y,
                   double *sr, int *best_a, int *best_k, double *depth)
{
    double bv = 0.0, bd = 0.0;
    int ba = 0, bk = kmin;
    for (int a = 0; a < nb; ++a) {
        double r = 0.0, s = 0.0;
        for (int k = 1; k <= kmax; ++k) {
            int j = (a + k - 1) % nb;
            r += W[j];
            s += Y[j];
            if (k < kmin) continue;
            double den = r * (1.0 - r);
            double v = (den > 0.0) ? (s * s) / den : 0.0;
            if (v > bv || (v == bv && v > 0.0 && (k < bk || (k == bk && a < ba)))) {
                bv = v; ba = a; bk = k; bd = s / den;
            }
        }
    }
    *sr = bv; *best_a = ba; *best_k = bk; *depth = bd;
}

/* O1..O4 for one curve over a frequency list.  Outputs have nf entries each.
 * Returns the status of oracle_prepare; on a data fault the outputs are zero-filled. */
int oracle_spectrum(int64_t n, const float *t, const float *mag, const float *sigma,
                    int64_t nf, const double *freqs, int nb, int kmin, int kmax,
                    double *sr, int32_t *best_a, int32_t *best_k, double *depth)
{
    double *w = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    double *x = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    double *W = (double *)malloc(sizeof(double) * (size_t)nb);
    double *Y = (double *)malloc(sizeof(double) * (size_t)nb);
    int st = oracle_prepare(n, t, mag, sigma, w, x);
    for (int64_t q = 0; q < nf; ++q) {
        if (st != 0) { sr[q] = 0.0; best_a[q] = 0; best_k[q] = kmin; depth[q] = 0.0; continue; }
        fold(n, t, w, x, freqs[q], nb, W, Y);
        int a, k;
        search(nb, kmin, kmax, W, Y, &sr[q], &a, &k, &depth[q]);
        best_a[q] = a; best_k[q] = k;
    }
    free(w); free(x); free(W); free(Y);
    return st;
}

/* O4 for a single box (a, k) at one frequency: used by the comparator to score the box the CUDA
 * path chose.  Returns SR (0 for an invalid box); *depth = s/(r(1-r)) or 0. */
double oracle_sr_at(int64_t n, const float *t, const float *mag, const float *sigma,
                    double f, int nb, int a, int k, double *depth)
{
    double *w = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    double *x = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    double *W = (double *)malloc(sizeof(double) * (size_t)nb);
    double *Y = (double *)malloc(sizeof(double) * (size_t)nb);
    double v = 0.0, d = 0.0;
    if (oracle_prepare(n, t, mag, sigma, w, x) == 0) {
        fold(n, t, w, x, f, nb, W, Y);
        double r = 0.0, s = 0.0;
        for (int kk = 1; kk <= k; ++kk) {
            int j = (a + kk - 1) % nb;
            r += W[j];
            s += Y[j];
        }
        double den = r * (1.0 - r);
        if (den > 0.0) { v = (s * s) / den; d = s / den; }
    }
    if (depth) *depth = d;
    free(w); free(x); free(W); free(Y);
    return v;
}

/* Folded bins at one frequency (for the tests that pin the fold itself). */
int oracle_fold_bins(int64_t n, const float *t, const float *mag, const float *sigma,
                     double f, int nb, double *W, double *Y)
{
    double *w = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    double *x = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    int st = oracle_prepare(n, t, mag, sigma, w, x);
    if (st == 0) fold(n, t, w, x, f, nb, W, Y);
    free(w); free(x);
    return st;
}

/* O5 (reading R14): index q is a peak iff SR[q] > 0 and (q == 0 or SR[q] > SR[q-1]) and
 * (q == nf-1 or SR[q] >= SR[q+1]); peaks are ranked by (SR descending, index ascending); the first
 * kpk are written to idx[], padded with -1.  Returns the number of peaks written. */
int oracle_peaks(int64_t nf, const double *sr, int kpk, int64_t *idx)
{
    int found = 0;
    for (int j = 0; j < kpk; ++j) idx[j] = -1;
    for (int64_t q = 0; q < nf; ++q) {
        if (!(sr[q] > 0.0)) continue;
        if (q > 0 && !(sr[q] > sr[q - 1])) continue;
        if (q < nf - 1 && !(sr[q] >= sr[q + 1])) continue;
        /* insert into the ranked list: strictly larger SR goes first; equal SR keeps index order */
        int pos = found < kpk ? found : kpk;
        while (pos > 0 && sr[q] > sr[idx[pos - 1]]) --pos;
        if (pos >= kpk) continue;
        int last = found < kpk ? found : kpk - 1;
        for (int j = last; j > pos; --j) idx[j] = idx[j - 1];
        idx[pos] = q;
        if (found < kpk) ++found;
    }
    return found;
}

/* Reading R14 with a minimum separation (SURVEY.md section 8(c) reading 14, the optional `peak_min_sep`): on a
 * fine grid the highest local maxima around one signal are its own sidelobes, and a list of candidates (PAPER.md
 * L151) should not spend every slot on one of them.  Exact greedy rule: walk ALL peaks of O5 in (SR descending,
 * index ascending) order; accept a peak iff its index is MORE than min_sep grid steps from every peak accepted so
 * far; stop at kpk.  A rejected peak suppresses nothing.  min_sep = 0 is oracle_peaks.  Returns the number written;
 * idx[] is padded with -1. */
int oracle_peaks_sep(int64_t nf, const double *sr, int kpk, int64_t min_sep, int64_t *idx)
{
    for (int j = 0; j < kpk; ++j) idx[j] = -1;
    int64_t *pk = (int64_t *)malloc(sizeof(int64_t) * (size_t)(nf > 0 ? nf : 1));
    int64_t np = 0;
    for (int64_t q = 0; q < nf; ++q) {                      /* the peaks of O5, in index order */
        if (!(sr[q] > 0.0)) continue;
        if (q > 0 && !(sr[q] > sr[q - 1])) continue;
        if (q < nf - 1 && !(sr[q] >= sr[q + 1])) continue;
        pk[np++] = q;
    }
    int found = 0;
    unsigned char *used = (unsigned char *)calloc((size_t)(np > 0 ? np : 1), 1);
    while (found < kpk) {
        /* the best peak not yet visited: largest SR, then smallest index (pk[] is in index order) */
        int64_t b = -1;
        for (int64_t i = 0; i < np; ++i)
            if (!used[i] && (b < 0 || sr[pk[i]] > sr[pk[b]])) b = i;
        if (b < 0) break;
        used[b] = 1;
        int far = 1;
        for (int j = 0; j < found; ++j) {
            int64_t d = pk[b] - idx[j];
            if (d < 0) d = -d;
            if (d <= min_sep) far = 0;
        }
        if (far) idx[found++] = pk[b];
    }
    free(pk); free(used);
    return found;
}

/* oracle_bin over arrays (for the bin-index parity test on very many (f, t) pairs). */
void oracle_bins_many(int64_t n, const double *f, const double *t, int nb, int32_t *bins)
{
    for (int64_t i = 0; i < n; ++i) bins[i] = oracle_bin(f[i], t[i], nb);
}

/* ---- f1: peak significance and refinement (readings S1-S4) ----
 * The paper calls its detections "high-confidence" candidates and names the BLS of
 * Kovacs et al. (L135) without printing a formula; these are the readings:
 *   S1  significance ("signal detection efficiency"): SDE(q) = (SR[q] - mean(SR)) / sd(SR), mean and
 *       POPULATION standard deviation over all nf samples of the curve's spectrum (the squared form R1);
 *       0 if sd = 0;
 *   S2  fine re-search around a peak at coarse index q: n_fine frequencies f_j = f_lo + j * step,
 *       step = (f_hi - f_lo)/(n_fine - 1), f_lo = freqs[max(q-1, 0)], f_hi = freqs[min(q+1, nf-1)]
 *       (n_fine = 1: f_0 = f_lo); each f_j evaluated in fp64 without contraction;
 *   S3  sub-bin phase resolution: the bin grid is shifted by s_h = h / (n_shift * nb) cycles,
 *       h = 0 .. n_shift-1: b = floor(nb * frac(f t - s_h)), by the rule of oracle_bin_shift;
 *   S4  the refined peak is the best box over (j, h), ties to the smallest j, then the smallest h;
 *       its box covers true phases [(a/nb + s_h), ((a+k)/nb + s_h)). */

/* S1 */
double oracle_sde(int64_t nf, const double *sr, int64_t q)
{
    double mean = 0.0;
    for (int64_t i = 0; i < nf; ++i) mean += sr[i];
    mean /= (double)nf;
    double var = 0.0;
    for (int64_t i = 0; i < nf; ++i) var += (sr[i] - mean) * (sr[i] - mean);
    double sd = sqrt(var / (double)nf);
    return sd > 0.0 ? (sr[q] - mean) / sd : 0.0;
}

/* S3: the phase rule R8 with the bin grid shifted by `shift` cycles: four individually rounded operations.
 *   p = RN(f*t) ; p2 = RN(p - shift) ; phi = p2 - floor(p2) (exact) ; b = trunc(RN(phi*nb)), clamped. */
int oracle_bin_shift(double f, double t, int nb, double shift)
{
    volatile double p = f * t;
    volatile double p2 = p - shift;
    double phi = p2 - floor(p2);
    volatile double xb = phi * (double)nb;
    int b = (int)xb;
    if (b >= nb) b = nb - 1;
    return b;
}

/* oracle_bin_shift over arrays, one shift for all pairs (for the shifted bin-index parity test on very many
 * (f, t) pairs): a loop around the rule above, nothing else. */
void oracle_bins_shift_many(int64_t n, const double *f, const double *t, int nb, double shift, int32_t *bins)
{
    for (int64_t i = 0; i < n; ++i) bins[i] = oracle_bin_shift(f[i], t[i], nb, shift);
}

/* S2 + S3: the spectrum of one curve on the fine grid, entry (j, h) at index j*n_shift + h. */
int oracle_refine_spectrum(int64_t n, const float *t, const float *mag, const float *sigma, double f_lo, double f_hi,
                           int n_fine, int n_shift, int nb, int kmin, int kmax,
                           double *freq, double *sr, int32_t *best_a, int32_t *best_k, double *depth)
{
    double *w = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    double *x = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    double *W = (double *)malloc(sizeof(double) * (size_t)nb);
    double *Y = (double *)malloc(sizeof(double) * (size_t)nb);
    int st = oracle_prepare(n, t, mag, sigma, w, x);
    volatile double step = n_fine > 1 ? (f_hi - f_lo) / (double)(n_fine - 1) : 0.0;
    for (int j = 0; j < n_fine; ++j) {
        volatile double js = (double)j * step;
        double f = f_lo + js;
        for (int h = 0; h < n_shift; ++h) {
            int64_t q = (int64_t)j * n_shift + h;
            freq[q] = f;
            if (st != 0) { sr[q] = 0.0; best_a[q] = 0; best_k[q] = kmin; depth[q] = 0.0; continue; }
            double shift = (double)h / (double)(n_shift * nb);
            for (int b = 0; b < nb; ++b) { W[b] = 0.0; Y[b] = 0.0; }
            for (int64_t i = 0; i < n; ++i) {
                int b = oracle_bin_shift(f, (double)t[i], nb, shift);
                W[b] += w[i];
                Y[b] += w[i] * x[i];
            }
            int a, k;
            search(nb, kmin, kmax, W, Y, &sr[q], &a, &k, &depth[q]);
            best_a[q] = a; best_k[q] = k;
        }
    }
    free(w); free(x); free(W); free(Y);
    return st;
}

/* S4: index of the refined peak in a fine spectrum of m = n_fine*n_shift entries: the largest SR, ties
 * to the smallest index (j major, h minor); -1 if every entry is 0. */
int64_t oracle_refine_pick(int64_t m, const double *sr)
{
    int64_t best = -1;
    double bv = 0.0;
    for (int64_t q = 0; q < m; ++q)
        if (sr[q] > bv) { bv = sr[q]; best = q; }
    return best;
}

/* ---- f4: eclipse detection efficiency of a cadence (Fig. 13) ----
 * "The detection efficiency is the probability that at least two eclipses will be observed from an
 * eclipsing target with a specified period, after observing window and weather effects have been taken into
 * account" -- "based on simulations including the actual observing cadences of the survey".  Readings:
 *   W1  the cadence is the list of epochs t_i of one light curve, sorted ascending (window and weather are
 *       whatever made that list);
 *   W2  a target of frequency f (period 1/f) and eclipse duration d days has mid-eclipse phase phi, uniform in
 *       [0, 1); the simulation takes the n_phase phases phi_k = (k + 1/2)/n_phase (a stratified grid: no
 *       random numbers, so both implementations see the same targets);
 *   W3  epoch t_i is in eclipse iff |x - rint(x)| <= h, x = RN(RN(f t_i) - phi_k), h = RN(RN(0.5 d) f)
 *       (rint = round half to even); the eclipse it belongs to is cycle m = rint(x);
 *   W4  an eclipse is "observed" if at least one epoch is inside it; the target is detected iff at least
 *       min_events DISTINCT cycles are observed (the paper: two); efficiency = detected phases / n_phase.
 * count[q] receives the number of detected phases at freqs[q], eff[q] = count / n_phase. */
void oracle_detection_efficiency(int64_t n, const float *t, int64_t nf, const double *freqs, double duration,
                                 int n_phase, int min_events, int32_t *count, double *eff)
{
    for (int64_t q = 0; q < nf; ++q) {
        const double f = freqs[q];
        volatile double hd = 0.5 * duration;
        volatile double h = hd * f;
        int32_t det = 0;
        for (int k = 0; k < n_phase; ++k) {
            const double phi = ((double)k + 0.5) / (double)n_phase;
            int events = 0;
            double last = 0.0;
            for (int64_t i = 0; i < n; ++i) {
                volatile double u = f * (double)t[i];
                volatile double x = u - phi;
                double m = rint(x);
                if (fabs(x - m) <= h && (events == 0 || m != last)) { ++events; last = m; }
            }
            if (events >= min_events) ++det;
        }
        count[q] = det;
        eff[q] = (double)det / (double)n_phase;
    }
}
