/*
 * umi_oracle.c -- fp64 CPU oracle for the UMI sliding-window estimator.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this
 * file.  It shares no code, header, table or helper with the CUDA path under
 * paper_2604_06602_b200/csrc/ and neither includes the other.
 *
 * What it is: the algorithm of PAPER.md section 2 written out per window, step
 * by step, in the paper's order and notation, in double precision, with no
 * sliding trick, no blocking and no fusion:
 *   window rule        PAPER.md:35   W = floor(0.5/dt) | 1
 *   Phase 1 median     PAPER.md:39   exact sample median (here: full sort, pick rank)
 *   Phase 2 upper-RMS  PAPER.md:43-48 (Eq. 1), s = 0.6745 * sigma_upper
 *   Phase 3 iterations PAPER.md:54-63 (Eq. 2-4), c = 5, alpha = 2, 5 passes
 *   minimum length     PAPER.md:192  W/3
 * Where the paper is silent the readings R1..R18 of DESIGN.md ("Readings of the
 * paper") are taken; each is marked (Rn) at the line that implements it.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): the paper-printed window
 * lengths and weight values, a hand-computed worked example, an independent
 * numpy brute force (oracle/brute.py), numpy/scipy median and mean routines,
 * the Gaussian closed forms, and the invariants listed in DESIGN.md.
 * Parity unpinned: none of the functions below; the paper's real-data accuracy
 * tables are out of scope and are not reproduced.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (no -ffast-math), see oracle/build.py.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define UMI_ORACLE_SCALE_CONST 0.6745

/* Sibling estimators on the same window machinery. */
#define UMI_ORACLE_SCALE_UPPER_RMS 0   /* PAPER.md:43-48, the paper's scale */
#define UMI_ORACLE_SCALE_MAD 1         /* the standard MAD (ablation) */
#define UMI_ORACLE_WEIGHT_BISQUARE 0   /* PAPER.md:58, Eq. 3 */
#define UMI_ORACLE_WEIGHT_WELSCH 1     /* Gaussian-shaped weights */

/* W = floor(0.5/dt) | 1, dt in days.
 * (R15) the quotient is nudged up by 2^-20 relative before the floor so that a
 * cadence that passed through fp32 (0.5/dt = 359.99999) still gives the
 * paper's 361.  Returns 0 for dt <= 0 or non-finite. */
int umi_oracle_window_len(double dt_days)
{
    if (!(dt_days > 0.0) || !isfinite(dt_days)) return 0;
    double q = (0.5 / dt_days) * (1.0 + ldexp(1.0, -20));
    if (!(q < 2147483646.0)) return 0;
    int w = (int)floor(q);
    return w | 1;
}

/* PAPER.md:56-58, Eq. 2 and Eq. 3: weight of a standardized residual u. */
double umi_oracle_weight(double u, double alpha)
{
    double ueff = (u < 0.0) ? alpha * u : u;          /* Eq. 2 (R13: u < 0) */
    if (fabs(ueff) < 1.0) {                            /* Eq. 3 (R12: strict) */
        double t = 1.0 - ueff * ueff;
        return t * t;
    }
    return 0.0;
}

static int cmp_double(const void *a, const void *b)
{
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

/* (R3, R16) a slot is valid iff it is inside the series, its flux is finite
 * and, when a time array is given, its time stamp is finite. */
static int slot_valid(const double *time, const float *flux, int64_t N, int64_t j)
{
    if (j < 0 || j >= N) return 0;                    /* (R2) edges truncate */
    if (!isfinite(flux[j])) return 0;
    if (time && !isfinite(time[j])) return 0;
    return 1;
}

/*
 * The estimator on the n valid samples x[0..n) of one window.
 * own_valid = the position's own slot is valid.  Outputs (any may be NULL): trend
 * (double), median (float), scale s, n_plus, near_cutoff flag.  sorted[] must
 * hold n doubles.  Returns 1 if a trend value was produced, 0 if the output is NaN.
 */
static int oracle_location_family(const double *x, int n, int own_valid,
                           int scale_kind, int weight_kind,
                           double alpha, double c, int n_iter, int min_valid,
                           double cutoff_tol, double *sorted,
                           double *trend, float *median, double *scale,
                           int32_t *n_plus_out, uint8_t *near_cutoff)
{
    if (trend) *trend = NAN;
    if (median) *median = NAN;
    if (scale) *scale = NAN;
    if (n_plus_out) *n_plus_out = 0;
    if (near_cutoff) *near_cutoff = 0;

    /* (R4) PAPER.md:192 minimum length W/3; (R5) invalid own slot -> NaN */
    if (!own_valid || n < min_valid || n < 1) return 0;

    /* Phase 1: the exact sample median.  Definition written out:
     * sort ascending, take rank k = (n-1)/2 (R6: lower middle when n is even). */
    memcpy(sorted, x, (size_t)n * sizeof(double));
    qsort(sorted, (size_t)n, sizeof(double), cmp_double);
    const double med = sorted[(n - 1) / 2];
    if (median) *median = (float)med;                 /* a selected fp32 sample: exact */

    double s;
    if (scale_kind == UMI_ORACLE_SCALE_MAD) {
        /* Sibling scale (F4): the standard MAD, the median of the absolute
         * deviations from the median, both sides.  (R21) rank (n-1)/2 of the sorted deviations,
         * as for the median itself (R6); used as s directly -- PAPER.md:48 scales sigma_upper
         * by 0.6745 "to match the MAD convention", so the MAD itself carries no factor. */
        for (int j = 0; j < n; ++j) sorted[j] = fabs(x[j] - med);
        qsort(sorted, (size_t)n, sizeof(double), cmp_double);
        s = sorted[(n - 1) / 2];
    } else {
    /* Phase 2, Eq. 1: RMS of residuals strictly above the median (R7). */
    int n_plus = 0;
    double ss = 0.0;
    for (int j = 0; j < n; ++j)
        if (x[j] > med) { double r = x[j] - med; ss += r * r; ++n_plus; }
    if (n_plus_out) *n_plus_out = n_plus;
    if (n_plus == 0) {                                /* (R8) */
        if (trend) *trend = med;
        if (scale) *scale = 0.0;
        return 1;
    }
    const double sigma_upper = sqrt(ss / (double)n_plus);
    s = UMI_ORACLE_SCALE_CONST * sigma_upper;
    }
    if (scale) *scale = s;
    if (!(s > 0.0)) {                                 /* (R8) */
        if (trend) *trend = med;
        return 1;
    }

    /* Phase 3: n_iter passes of Eq. 2-4, s held fixed (R9),
     * no convergence test (R10). */
    double mu = med;
    int flagged = 0;
    for (int it = 0; it < n_iter; ++it) {
        double sw = 0.0, swx = 0.0;
        for (int j = 0; j < n; ++j) {
            double u = (x[j] - mu) / (c * s);
            double ueff = (u < 0.0) ? alpha * u : u;  /* Eq. 2 */
            double w;
            if (weight_kind == UMI_ORACLE_WEIGHT_WELSCH) {
                /* Sibling weight (F4; "Welsch ... Gaussian-shaped weights"):
                 * (R22) w = exp(-u_eff^2), no cut-off. */
                w = exp(-ueff * ueff);
            } else {
            if (fabs(ueff) < 1.0) { double t = 1.0 - ueff * ueff; w = t * t; }   /* Eq. 3 */
            else w = 0.0;
            if (fabs(fabs(ueff) - 1.0) <= cutoff_tol) flagged = 1;
            }
            sw += w;
            swx += w * x[j];
        }
        if (!(sw > 0.0)) break;                       /* (R11) */
        mu = swx / sw;                                /* Eq. 4 */
    }
    if (trend) *trend = mu;
    if (near_cutoff) *near_cutoff = (uint8_t)flagged;
    return 1;
}

/* The paper's estimator: upper-RMS scale, bisquare weights. */
static int oracle_location(const double *x, int n, int own_valid,
                           double alpha, double c, int n_iter, int min_valid,
                           double cutoff_tol, double *sorted,
                           double *trend, float *median, double *scale,
                           int32_t *n_plus_out, uint8_t *near_cutoff)
{
    return oracle_location_family(x, n, own_valid, UMI_ORACLE_SCALE_UPPER_RMS, UMI_ORACLE_WEIGHT_BISQUARE,
                                  alpha, c, n_iter, min_valid, cutoff_tol, sorted,
                                  trend, median, scale, n_plus_out, near_cutoff);
}

/*
 * One window: star row (time, flux) of length N, position i.
 * Outputs (any may be NULL): trend (double), median (float), scale s, n valid,
 * n_plus, near_cutoff flag.  work[] must hold 2*W doubles.
 * Returns 1 if a trend value was produced, 0 if the output is NaN.
 */
static int oracle_window(const double *time, const float *flux, int64_t N, int64_t i,
                         int W, double alpha, double c, int n_iter, int min_valid,
                         double cutoff_tol, double *work,
                         double *trend, float *median, double *scale,
                         int32_t *n_valid, int32_t *n_plus_out, uint8_t *near_cutoff)
{
    const int64_t h = (W - 1) / 2;                    /* (R1) centred window [i-h, i+h] */
    double *x = work, *sorted = work + W;
    int n = 0;
    for (int64_t j = i - h; j <= i + h; ++j)
        if (slot_valid(time, flux, N, j)) x[n++] = (double)flux[j];   /* exact widening */
    if (n_valid) *n_valid = n;
    return oracle_location(x, n, slot_valid(time, flux, N, i), alpha, c, n_iter, min_valid,
                           cutoff_tol, sorted, trend, median, scale, n_plus_out, near_cutoff);
}

static int resolve_min_valid(int W, int min_valid)
{
    if (min_valid >= 0) return min_valid;
    int m = W / 3;                                    /* (R4) PAPER.md:192 */
    return m < 1 ? 1 : m;
}

/*
 * Evaluate a list of (star, position) pairs.  flux is [n_stars, n_cadences]
 * row-major fp32; time is NULL or the same shape in fp64.
 * min_valid < 0 selects the default max(1, W/3).
 * Every output array has `count` entries and may be NULL.
 * Returns 0 on success, 1 on invalid arguments.
 */
int umi_oracle_positions(const double *time, const float *flux,
                         int64_t n_stars, int64_t n_cadences,
                         const int64_t *star_idx, const int64_t *pos_idx, int64_t count,
                         int W, double alpha, double c, int n_iter, int min_valid,
                         double cutoff_tol,
                         double *trend64, float *trend32, float *median,
                         double *scale, int32_t *n_valid, int32_t *n_plus,
                         uint8_t *near_cutoff)
{
    if (!flux || n_stars < 0 || n_cadences < 0 || W < 1 || (W & 1) == 0 || n_iter < 0 ||
        !(alpha > 0.0) || !(c > 0.0) || count < 0)
        return 1;
    const int mv = resolve_min_valid(W, min_valid);
    int bad = 0;
#pragma omp parallel
    {
        double *work = (double *)malloc((size_t)2 * (size_t)W * sizeof(double));
#pragma omp for schedule(dynamic, 256)
        for (int64_t q = 0; q < count; ++q) {
            int64_t b = star_idx[q], i = pos_idx[q];
            if (!work || b < 0 || b >= n_stars || i < 0 || i >= n_cadences) {
#pragma omp atomic write
                bad = 1;
                continue;
            }
            const float *frow = flux + b * n_cadences;
            const double *trow = time ? time + b * n_cadences : NULL;
            double t64;
            oracle_window(trow, frow, n_cadences, i, W, alpha, c, n_iter, mv, cutoff_tol, work,
                          &t64, median ? median + q : NULL, scale ? scale + q : NULL,
                          n_valid ? n_valid + q : NULL, n_plus ? n_plus + q : NULL,
                          near_cutoff ? near_cutoff + q : NULL);
            if (trend64) trend64[q] = t64;
            if (trend32) trend32[q] = (float)t64;     /* round-to-nearest-even */
        }
        free(work);
    }
    return bad;
}

/* Every position of every star, in [n_stars, n_cadences] order. */
int umi_oracle_detrend(const double *time, const float *flux,
                       int64_t n_stars, int64_t n_cadences,
                       int W, double alpha, double c, int n_iter, int min_valid,
                       double cutoff_tol,
                       double *trend64, float *trend32, float *median,
                       double *scale, int32_t *n_valid, int32_t *n_plus,
                       uint8_t *near_cutoff)
{
    if (!flux || n_stars < 0 || n_cadences < 0 || W < 1 || (W & 1) == 0 || n_iter < 0 ||
        !(alpha > 0.0) || !(c > 0.0))
        return 1;
    const int mv = resolve_min_valid(W, min_valid);
    const int64_t total = n_stars * n_cadences;
    int bad = 0;
#pragma omp parallel
    {
        double *work = (double *)malloc((size_t)2 * (size_t)W * sizeof(double));
#pragma omp for schedule(dynamic, 256)
        for (int64_t q = 0; q < total; ++q) {
            if (!work) {
#pragma omp atomic write
                bad = 1;
                continue;
            }
            int64_t b = q / n_cadences, i = q % n_cadences;
            const float *frow = flux + b * n_cadences;
            const double *trow = time ? time + b * n_cadences : NULL;
            double t64;
            oracle_window(trow, frow, n_cadences, i, W, alpha, c, n_iter, mv, cutoff_tol, work,
                          &t64, median ? median + q : NULL, scale ? scale + q : NULL,
                          n_valid ? n_valid + q : NULL, n_plus ? n_plus + q : NULL,
                          near_cutoff ? near_cutoff + q : NULL);
            if (trend64) trend64[q] = t64;
            if (trend32) trend32[q] = (float)t64;
        }
        free(work);
    }
    return bad;
}

/*
 * Normalisation stage ("detrending, normalization"): flat = flux / trend,
 * one division per cadence in fp64 (fp32 flux widened exactly); NaN where trend is NaN.
 */
int umi_oracle_normalize(const float *flux, const double *trend64, int64_t count, double *flat64)
{
    if (!flux || !trend64 || !flat64 || count < 0) return 1;
    for (int64_t q = 0; q < count; ++q) flat64[q] = (double)flux[q] / trend64[q];
    return 0;
}

/*
 * Gap handling by time stamps ("gap handling"; reading R20): the
 * rows are COMPACTED series (cadences were removed, so time jumps) of n_samples samples
 * with real time stamps.  Sample (b, i) sits in slot k_i = rint((time[i] - t0) / dt)
 * (round half to even) of a uniform grid of n_grid slots; it is valid iff time and flux
 * are finite, 0 <= k_i < n_grid, and the NEXT sample of the row does not map to the same
 * slot.  Its window is the valid samples j of the same row with |k_j - k_i| <= h: W slots
 * of fixed duration W*dt, exactly what the positional window of PAPER.md:35 spans on an
 * uncompacted series.  Times are assumed non-decreasing along a row, so only samples
 * j in [i-h, i+h] can qualify.  Outputs as umi_oracle_detrend, [n_stars, n_samples].
 */
int umi_oracle_gapped(const double *time, const float *flux,
                      int64_t n_stars, int64_t n_samples,
                      double t0, double dt, int64_t n_grid,
                      int W, double alpha, double c, int n_iter, int min_valid,
                      double cutoff_tol,
                      double *trend64, float *trend32, float *median,
                      double *scale, int32_t *n_valid, int32_t *n_plus,
                      uint8_t *near_cutoff)
{
    if (!time || !flux || n_stars < 0 || n_samples < 0 || n_grid < 0 || W < 1 || (W & 1) == 0 ||
        n_iter < 0 || !(alpha > 0.0) || !(c > 0.0) || !(dt > 0.0) || !isfinite(dt) || !isfinite(t0))
        return 1;
    const int mv = resolve_min_valid(W, min_valid);
    const int64_t h = (W - 1) / 2;
    const int64_t total = n_stars * n_samples;
    int64_t *slot = (int64_t *)malloc((size_t)(total > 0 ? total : 1) * sizeof(int64_t));
    if (!slot) return 1;
    /* slot of every sample, -1 = invalid */
    for (int64_t b = 0; b < n_stars; ++b) {
        const double *trow = time + b * n_samples;
        const float *frow = flux + b * n_samples;
        int64_t *srow = slot + b * n_samples;
        for (int64_t i = 0; i < n_samples; ++i) {
            srow[i] = -1;
            if (!isfinite(trow[i])) continue;
            double k = rint((trow[i] - t0) / dt);
            if (!(k >= 0.0) || !(k < (double)n_grid)) continue;
            srow[i] = (int64_t)k;
        }
        for (int64_t i = 0; i < n_samples; ++i) {
            int64_t k = srow[i];
            /* a sample that shares its slot with its successor is dropped */
            if (k >= 0 && i + 1 < n_samples && isfinite(trow[i + 1])) {
                double kn = rint((trow[i + 1] - t0) / dt);
                if (kn == (double)k) srow[i] = -1;
            }
        }
        for (int64_t i = 0; i < n_samples; ++i)
            if (!isfinite(frow[i])) srow[i] = -1;
    }
    int bad = 0;
#pragma omp parallel
    {
        double *work = (double *)malloc((size_t)2 * (size_t)W * sizeof(double));
#pragma omp for schedule(dynamic, 256)
        for (int64_t q = 0; q < total; ++q) {
            if (!work) {
#pragma omp atomic write
                bad = 1;
                continue;
            }
            const int64_t b = q / n_samples, i = q % n_samples;
            const float *frow = flux + b * n_samples;
            const int64_t *srow = slot + b * n_samples;
            const int64_t ki = srow[i];
            int n = 0;
            if (ki >= 0) {
                for (int64_t j = i - h; j <= i + h; ++j) {
                    if (j < 0 || j >= n_samples || srow[j] < 0) continue;
                    int64_t d = srow[j] - ki;
                    if (d < 0) d = -d;
                    if (d <= h) work[n++] = (double)frow[j];
                }
            }
            if (n_valid) n_valid[q] = n;
            double t64;
            oracle_location(work, n, ki >= 0, alpha, c, n_iter, mv, cutoff_tol, work + W,
                            &t64, median ? median + q : NULL, scale ? scale + q : NULL,
                            n_plus ? n_plus + q : NULL, near_cutoff ? near_cutoff + q : NULL);
            if (trend64) trend64[q] = t64;
            if (trend32) trend32[q] = (float)t64;
        }
        free(work);
    }
    free(slot);
    return bad;
}

/*
 * Gap handling with segments (next row F2, second part; "gap handling", PAPER.md:192
 * "minimum segment length ... W/3"; reading R23).  On top of umi_oracle_gapped (R20):
 *   - the valid samples of a row, in order, are cut into SEGMENTS wherever more than break_slots
 *     empty slots lie between two consecutive valid samples (break_slots < 0: never);
 *   - a segment with fewer than min_segment valid samples is dropped: NaN out, in no window;
 *   - the window of a sample holds samples of its OWN segment only (|slot difference| <= h);
 *   - a sample whose slot lies less than edge_cut slots from the first or the last slot of its
 *     segment gets NaN out, but still takes part in the windows of the others.
 * break_slots < 0, min_segment <= 0, edge_cut <= 0 is umi_oracle_gapped.
 */
int umi_oracle_gapped_ex(const double *time, const float *flux,
                         int64_t n_stars, int64_t n_samples,
                         double t0, double dt, int64_t n_grid,
                         int W, double alpha, double c, int n_iter, int min_valid,
                         int64_t break_slots, int64_t min_segment, int64_t edge_cut,
                         double cutoff_tol,
                         double *trend64, float *trend32, float *median,
                         double *scale, int32_t *n_valid, int32_t *n_plus,
                         uint8_t *near_cutoff)
{
    if (!time || !flux || n_stars < 0 || n_samples < 0 || n_grid < 0 || W < 1 || (W & 1) == 0 ||
        n_iter < 0 || !(alpha > 0.0) || !(c > 0.0) || !(dt > 0.0) || !isfinite(dt) || !isfinite(t0))
        return 1;
    const int mv = resolve_min_valid(W, min_valid);
    const int64_t h = (W - 1) / 2;
    const int64_t total = n_stars * n_samples;
    const size_t cnt = (size_t)(total > 0 ? total : 1);
    int64_t *slot = (int64_t *)malloc(cnt * sizeof(int64_t));   /* -1 = invalid */
    int64_t *seg = (int64_t *)malloc(cnt * sizeof(int64_t));    /* segment number inside the row, -1 = none */
    uint8_t *cut = (uint8_t *)malloc(cnt);                       /* 1 = inside the edge cut */
    if (!slot || !seg || !cut) { free(slot); free(seg); free(cut); return 1; }
    for (int64_t b = 0; b < n_stars; ++b) {
        const double *trow = time + b * n_samples;
        const float *frow = flux + b * n_samples;
        int64_t *srow = slot + b * n_samples, *grow = seg + b * n_samples;
        uint8_t *crow = cut + b * n_samples;
        /* (R20) slot of every sample, as in umi_oracle_gapped */
        for (int64_t i = 0; i < n_samples; ++i) {
            srow[i] = -1;
            if (!isfinite(trow[i])) continue;
            double k = rint((trow[i] - t0) / dt);
            if (!(k >= 0.0) || !(k < (double)n_grid)) continue;
            srow[i] = (int64_t)k;
        }
        for (int64_t i = 0; i < n_samples; ++i) {
            int64_t k = srow[i];
            if (k >= 0 && i + 1 < n_samples && isfinite(trow[i + 1])) {
                double kn = rint((trow[i + 1] - t0) / dt);
                if (kn == (double)k) srow[i] = -1;
            }
        }
        for (int64_t i = 0; i < n_samples; ++i)
            if (!isfinite(frow[i])) srow[i] = -1;
        /* (R23) segments: a new one starts after more than break_slots empty slots */
        int64_t cur = -1, prev_slot = 0;
        for (int64_t i = 0; i < n_samples; ++i) {
            grow[i] = -1;
            crow[i] = 0;
            if (srow[i] < 0) continue;
            if (cur < 0 || (break_slots >= 0 && srow[i] - prev_slot - 1 > break_slots)) ++cur;
            grow[i] = cur;
            prev_slot = srow[i];
        }
        /* per segment: count, first and last slot; short segments dropped, edges marked */
        for (int64_t i = 0; i < n_samples;) {
            if (grow[i] < 0) { ++i; continue; }
            int64_t j = i, last = i, count = 0;
            for (; j < n_samples; ++j) {
                if (grow[j] < 0) continue;
                if (grow[j] != grow[i]) break;
                ++count;
                last = j;
            }
            if (min_segment > 0 && count < min_segment) {
                for (int64_t m = i; m <= last; ++m)
                    if (grow[m] == grow[i]) { srow[m] = -1; }
                for (int64_t m = i; m <= last; ++m)
                    if (srow[m] < 0) grow[m] = -1;
            } else if (edge_cut > 0) {
                for (int64_t m = i; m <= last; ++m)
                    if (grow[m] >= 0 && (srow[m] - srow[i] < edge_cut || srow[last] - srow[m] < edge_cut)) crow[m] = 1;
            }
            i = j;
        }
    }
    int bad = 0;
#pragma omp parallel
    {
        double *work = (double *)malloc((size_t)2 * (size_t)W * sizeof(double));
#pragma omp for schedule(dynamic, 256)
        for (int64_t q = 0; q < total; ++q) {
            if (!work) {
#pragma omp atomic write
                bad = 1;
                continue;
            }
            const int64_t b = q / n_samples, i = q % n_samples;
            const float *frow = flux + b * n_samples;
            const int64_t *srow = slot + b * n_samples, *grow = seg + b * n_samples;
            const int64_t ki = srow[i];
            int n = 0;
            if (ki >= 0) {
                for (int64_t j = i - h; j <= i + h; ++j) {
                    if (j < 0 || j >= n_samples || srow[j] < 0 || grow[j] != grow[i]) continue;
                    int64_t d = srow[j] - ki;
                    if (d < 0) d = -d;
                    if (d <= h) work[n++] = (double)frow[j];
                }
            }
            if (n_valid) n_valid[q] = n;
            double t64;
            oracle_location(work, n, ki >= 0 && !cut[q], alpha, c, n_iter, mv, cutoff_tol, work + W,
                            &t64, median ? median + q : NULL, scale ? scale + q : NULL,
                            n_plus ? n_plus + q : NULL, near_cutoff ? near_cutoff + q : NULL);
            if (trend64) trend64[q] = t64;
            if (trend32) trend32[q] = (float)t64;
        }
        free(work);
    }
    free(slot);
    free(seg);
    free(cut);
    return bad;
}

/*
 * Sibling estimators (F4): every position of every star with the chosen scale and weight.
 * scale_kind 0 / weight_kind 0 is umi_oracle_detrend.  n_plus is not produced for the MAD.
 */
int umi_oracle_family(const double *time, const float *flux,
                      int64_t n_stars, int64_t n_cadences,
                      int W, int scale_kind, int weight_kind,
                      double alpha, double c, int n_iter, int min_valid, double cutoff_tol,
                      double *trend64, float *trend32, float *median,
                      double *scale, int32_t *n_valid, int32_t *n_plus,
                      uint8_t *near_cutoff)
{
    if (!flux || n_stars < 0 || n_cadences < 0 || W < 1 || (W & 1) == 0 || n_iter < 0 ||
        !(alpha > 0.0) || !(c > 0.0) || scale_kind < 0 || scale_kind > 1 || weight_kind < 0 || weight_kind > 1)
        return 1;
    const int mv = resolve_min_valid(W, min_valid);
    const int64_t h = (W - 1) / 2;
    const int64_t total = n_stars * n_cadences;
    int bad = 0;
#pragma omp parallel
    {
        double *work = (double *)malloc((size_t)2 * (size_t)W * sizeof(double));
#pragma omp for schedule(dynamic, 256)
        for (int64_t q = 0; q < total; ++q) {
            if (!work) {
#pragma omp atomic write
                bad = 1;
                continue;
            }
            const int64_t b = q / n_cadences, i = q % n_cadences;
            const float *frow = flux + b * n_cadences;
            const double *trow = time ? time + b * n_cadences : NULL;
            int n = 0;
            for (int64_t j = i - h; j <= i + h; ++j)
                if (slot_valid(trow, frow, n_cadences, j)) work[n++] = (double)frow[j];
            if (n_valid) n_valid[q] = n;
            double t64;
            oracle_location_family(work, n, slot_valid(trow, frow, n_cadences, i), scale_kind, weight_kind,
                                   alpha, c, n_iter, mv, cutoff_tol, work + W,
                                   &t64, median ? median + q : NULL, scale ? scale + q : NULL,
                                   n_plus ? n_plus + q : NULL, near_cutoff ? near_cutoff + q : NULL);
            if (trend64) trend64[q] = t64;
            if (trend32) trend32[q] = (float)t64;
        }
        free(work);
    }
    return bad;
}

int umi_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
