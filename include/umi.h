/*
 * umi.h -- C ABI of the B200 (sm_100a) UMI sliding-window detrender.
 *
 * UMI = the sliding-window asymmetric robust location estimator of
 * arxiv/paper_2604_06602, section 2 (lines 33-63):
 *   window rule   PAPER.md:35     W = floor(0.5/dt) | 1
 *   Phase 1       PAPER.md:37-39  exact sample median of the window
 *   Phase 2       PAPER.md:41-50  upper-RMS scale, Eq. 1, s = 0.6745 * sigma_upper
 *   Phase 3       PAPER.md:52-63  n_iter asymmetric Tukey-bisquare passes, Eq. 2-4, c = 5
 *   min. length   PAPER.md:192    fewer than max(1, W/3) valid samples -> NaN
 * Readings of everything the paper leaves open (edges, gaps, even counts,
 * ties, degenerate scale): DESIGN.md, "Readings of the paper", R1..R18.
 *
 * Conventions
 *  - Every entry point returns a umi_status (int); nothing throws or aborts
 *    across this boundary.  Arguments are validated on the host before any
 *    work is enqueued.
 *  - No torch types.  The DEVICE entry points allocate nothing, create nothing and keep
 *    no state: the only scratch their kernels share is trend_out itself, and any further
 *    buffer is a caller-owned workspace (umi_detrend_gapped).  They are re-entrant and may
 *    be called concurrently from several host threads on different streams.  The HOST
 *    batch driver (umi_detrend_host, umi_flatten_host) has to own device buffers and
 *    streams; it keeps them per device in a free list of slots (a stream and one buffer
 *    that is only ever grown; plain cudaMalloc, no memory pool of the device or of its
 *    own) for the next call, until umi_shutdown().  Nothing reads the process environment.
 *  - "DEVICE pointer": memory of the current CUDA device, readable/writable by
 *    kernels launched on `stream`.  "HOST pointer": ordinary host memory
 *    (pinned memory makes the copies asynchronous and faster, but is not
 *    required).
 *  - Layout: [n_stars, n_cadences] row-major, contiguous, row stride
 *    n_cadences elements, 64-bit indexing.
 *  - Invalid sample: flux not finite (NaN, +Inf, -Inf), or time given and not
 *    finite.  Invalid samples and slots outside [0, n_cadences) are skipped by
 *    every window (R2, R3, R16).
 *  - Reproducibility: a call is deterministic (no atomics on floating-point data), and the median is
 *    bit-exact always.  The trend of a star may differ in its last bits (~1e-7 relative) between calls
 *    with different batch sizes, because small batches run the split-window variant of the
 *    reweighting kernel, which sums the same terms in another order.
 *  - Supported dynamic range: the passes run on samples centred on one of the medians of
 *    the 128 consecutive positions a warp owns (4 for windows of at most 49 samples), the
 *    one of smallest magnitude, so the 1e-5 bar on the trend holds relative to the
 *    position's own |median| (for a light curve: the local flux); samples of any finite
 *    magnitude (fill values, glitches, whole runs of them) cost the others no precision.  (max - min) * 16 * max(1, 1/alpha) over the
 *    valid samples of those positions' windows must be finite in fp32.  Where the trend itself is a
 *    cancellation (a series already brought to zero mean, flux - 1) a bar relative to |trend| is not
 *    meaningful: the error there is bounded by 2e-6 of the typical |sample| of the window plus 1e-5 |trend|
 *    (measured: 3.5e-7 of it).
 */
#ifndef UMI_B200_H
#define UMI_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    UMI_OK = 0,
    UMI_ERR_INVALID_ARG = 1, /* null pointer, negative size, even or < 1 W, alpha/c not finite or <= 0, n_iter < 0 */
    UMI_ERR_UNSUPPORTED = 2, /* W > UMI_MAX_WINDOW */
    UMI_ERR_CUDA = 3,        /* launch / copy / allocation failure (the CUDA error is cleared) */
    UMI_ERR_TOO_LARGE = 4    /* umi_detrend_gapped_static: the job needs more than UMI_STATIC_SCRATCH_BYTES of scratch */
} umi_status;

/* Largest window the compiled kernels accept (TESS 20 s needs 2161). */
#define UMI_MAX_WINDOW 4097

/*
 * Window rule: W = floor(0.5/dt) | 1, dt = cadence in days.
 * (R15) the quotient is multiplied by (1 + 2^-20) before the floor so that a
 * cadence that passed through fp32 (0.5/dt = 359.99999) still gives 361.
 * Host only.  Returns W (odd, >= 1), or 0 if dt <= 0, non-finite, or W would
 * not fit an int.
 */
int umi_window_len(double dt_days);

/*
 * The hot path: trend_out[b, i] = UMI location of the centred window
 * [i-h, i+h], h = (W-1)/2, of star b, for every b and i.
 *
 *   time      DEVICE, const double [n_stars*n_cadences], or NULL.  Only
 *             finiteness is used: a non-finite time marks the cadence invalid.
 *   flux      DEVICE, const float [n_stars*n_cadences].
 *   n_stars, n_cadences   >= 0; either 0 -> UMI_OK, nothing enqueued.
 *   W         odd, 1 <= W <= UMI_MAX_WINDOW; may exceed n_cadences (clipped).
 *   alpha     asymmetry factor of Eq. 2 (2 = TESS default, 1 = symmetric); finite, > 0.
 *   n_iter    number of Eq. 2-4 passes (paper: 5); 0 returns the Phase-1
 *             median, bit-exact (it is a selected input sample; -0.0 reads as +0.0).
 *   trend_out DEVICE, float [n_stars*n_cadences]; must not overlap flux/time.
 *             NaN where the cadence itself is invalid or its window holds
 *             fewer than max(1, W/3) valid samples (R4, R5).  Also used as
 *             scratch between the two kernels of the call.
 *   stream    cudaStream_t (as void*), or NULL for the legacy default stream.
 *             Work is enqueued; the call does not synchronise.  The caller
 *             keeps all three buffers alive until the stream has drained.
 *
 * Scratch: none besides trend_out.  Between the two kernels of a call trend_out holds, per
 * position, where in its window the median sample sits and the count n+ of Eq. 1; the
 * second kernel overwrites both with the trend.  The call allocates nothing.
 *
 * c is fixed at 5.0.  Errors: see umi_status.
 */
int umi_detrend(const double* time, const float* flux,
                int64_t n_stars, int64_t n_cadences,
                int W, float alpha, int n_iter,
                float* trend_out, void* stream);

/*
 * Same path with the remaining parameters of PAPER.md Table 4 (lines 202-209)
 * exposed: tuning constant c (5.0 default, 2.5 "aggressive"; finite, > 0) and
 * min_valid (< 0 selects max(1, W/3)).  All pointers DEVICE.
 */
int umi_detrend_ex(const double* time, const float* flux,
                   int64_t n_stars, int64_t n_cadences,
                   int W, float alpha, float c, int n_iter, int min_valid,
                   float* trend_out, void* stream);

/*
 * Detrend + normalise ("detrending, normalization"): umi_detrend_ex, and in the
 * same kernels' epilogue flat_out[b, i] = flux[b, i] / trend_out[b, i] (one IEEE fp32
 * division; NaN wherever trend_out is NaN).  With n_iter = 0 the divisor is the median.
 *   flat_out  DEVICE, float [n_stars*n_cadences]; must not overlap the other buffers;
 *             NULL -> UMI_ERR_INVALID_ARG (use umi_detrend_ex).
 * trend_out is still required (it is the scratch between the kernels).
 */
int umi_flatten(const double* time, const float* flux,
                int64_t n_stars, int64_t n_cadences,
                int W, float alpha, float c, int n_iter, int min_valid,
                float* trend_out, float* flat_out, void* stream);

/*
 * Sibling estimators on the same window machinery: the scale and the
 * weight function are selectable; everything else (window, validity, median start, n_iter
 * passes of Eq. 2 + Eq. 4 with fixed s, c, alpha, min_valid) is umi_detrend_ex.
 *   scale_kind   UMI_SCALE_UPPER_RMS  Eq. 1, s = 0.6745 sigma_upper (the paper's scale)
 *                UMI_SCALE_MAD        s = median |x - median| over the window, both sides, the
 *                                     "standard MAD" of PAPER.md:50 / the ablation of PAPER.md:91;
 *                                     rank (n-1)/2 of the n deviations (R21), no extra factor
 *   weight_kind  UMI_WEIGHT_BISQUARE  Eq. 3
 *                UMI_WEIGHT_WELSCH    w = exp(-u_eff^2) ("Gaussian-shaped weights", R22)
 * alpha = 1 with the MAD and bisquare weights is the classic symmetric biweight location.
 *   scale_out  DEVICE, float [n_stars*n_cadences]: receives s per position (NaN where the trend
 *              is NaN).  REQUIRED for UMI_SCALE_MAD (it carries the MAD from the selection
 *              kernel to the reweighting kernel), optional (may be NULL) for the upper-RMS.
 *   flat_out   DEVICE or NULL: flux / trend as in umi_flatten.
 * Other arguments and errors as umi_detrend_ex; an unknown kind -> UMI_ERR_INVALID_ARG.
 */
#define UMI_SCALE_UPPER_RMS 0
#define UMI_SCALE_MAD 1
#define UMI_WEIGHT_BISQUARE 0
#define UMI_WEIGHT_WELSCH 1
int umi_detrend_family(const double* time, const float* flux,
                       int64_t n_stars, int64_t n_cadences,
                       int W, int scale_kind, int weight_kind,
                       float alpha, float c, int n_iter, int min_valid,
                       float* trend_out, float* scale_out, float* flat_out, void* stream);

/*
 * Gap handling by time stamps ("gap handling", the stage in front of the
 * detrender; reading R20).  The rows are COMPACTED series: cadences were removed
 * upstream, so time jumps.  Sample (b, i) sits in slot k = rint((time[b, i] - t0) / dt)
 * (fp64, round half to even) of a uniform grid of n_grid slots, and its window is the valid
 * samples of its row whose slot differs from k by at most h = (W-1)/2 -- the same W*dt of
 * time the positional window of PAPER.md:35 spans on an uncompacted row.  A sample is
 * invalid (NaN out, in no window) iff its time or flux is not finite, k is outside
 * [0, n_grid), or the next sample of its row lands in the same slot.  Rows must be
 * non-decreasing in time (otherwise the result is unspecified but memory-safe); rows
 * shorter than n_samples are padded with NaN time.
 *
 * Implementation: NaN-fill + scatter onto the grid, the hot path on [n_stars, n_grid],
 * gather back (csrc/umi_regrid.cu).
 *   time       DEVICE, const double [n_stars*n_samples]; required.
 *   flux       DEVICE, const float  [n_stars*n_samples].
 *   t0, dt     grid origin and cadence in the unit of `time`; dt > 0, both finite.
 *   n_grid     >= 0 slots per row (e.g. 1 + rint((t_last - t0)/dt)).
 *   trend_out  DEVICE, float [n_stars*n_samples].
 *   flat_out   DEVICE, float [n_stars*n_samples] or NULL: flux / trend.
 *   workspace  DEVICE, at least umi_gapped_workspace_bytes(n_stars, n_grid) bytes, owned by
 *              the caller, free to reuse once the stream has passed the call; too small or
 *              NULL -> UMI_ERR_INVALID_ARG.  It holds the two fp32 slot grids (flux, trend:
 *              8 bytes per slot): this entry point allocates nothing.
 * Enqueues on `stream`; does not synchronise.
 */
size_t umi_gapped_workspace_bytes(int64_t n_stars, int64_t n_grid);
int umi_detrend_gapped(const double* time, const float* flux,
                       int64_t n_stars, int64_t n_samples,
                       double t0, double dt, int64_t n_grid,
                       int W, float alpha, float c, int n_iter, int min_valid,
                       float* trend_out, float* flat_out,
                       void* workspace, size_t workspace_bytes, void* stream);

/*
 * The same with SEGMENTS (reading R23; "gap handling", "minimum
 * segment length ... W/3"): the valid samples of a row are cut into segments wherever more than
 * break_slots empty slots lie between two consecutive ones, and
 *   min_segment  a segment with fewer valid samples is dropped: NaN out, in no window (<= 0: off);
 *   edge_cut     samples less than edge_cut slots from the first or the last slot of their segment get
 *                NaN (trend and flat) but still take part in the windows of the others (<= 0: off);
 *   break_slots  < 0: the row is one segment.  Windows are never clipped at a break, which is exact
 *                whenever no window can reach across one: break_slots >= (W-1)/2 is required,
 *                0 <= break_slots < (W-1)/2 -> UMI_ERR_UNSUPPORTED.  (For a break of half a day on a
 *                half-day window, the usual choice, break_slots = W - 1.)
 * With all three off this is umi_detrend_gapped.  Needs umi_gapped_ex_workspace_bytes (17 bytes per
 * slot) when any of them is on, else umi_gapped_workspace_bytes; n_grid <= 2^31 - 1.
 */
size_t umi_gapped_ex_workspace_bytes(int64_t n_stars, int64_t n_grid);
int umi_detrend_gapped_ex(const double* time, const float* flux,
                          int64_t n_stars, int64_t n_samples,
                          double t0, double dt, int64_t n_grid,
                          int W, float alpha, float c, int n_iter, int min_valid,
                          int64_t break_slots, int64_t min_segment, int64_t edge_cut,
                          float* trend_out, float* flat_out,
                          void* workspace, size_t workspace_bytes, void* stream);

/*
 * umi_detrend_gapped_ex for callers that cannot allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc) and so have no workspace to pass: the scratch is a fixed array
 * of UMI_STATIC_SCRATCH_BYTES (16 MiB) of device memory inside the library's image, which every GPU that
 * loads the library holds until the process exits.  Same arguments (all pointers DEVICE, caller-owned
 * inputs and outputs), same kernels and same results as umi_detrend_gapped_ex; no cudaMalloc, cudaFree or
 * allocating library routine is called, now or later.
 *   Limit     n_stars * n_grid * 8 bytes (17 with any of break_slots / min_segment / edge_cut on) must not
 *             exceed UMI_STATIC_SCRATCH_BYTES: 2,097,152 slots (e.g. 100 stars x 20,971 slots), 986,895 with
 *             segments.  Beyond it -> UMI_ERR_TOO_LARGE, nothing enqueued (use umi_detrend_gapped_ex).
 *   Sharing   every call on a device uses the same array, which keeps the last call's contents.  The path
 *             clears what it needs first thing on `stream`, so calls ordered one after another (one stream,
 *             or streams ordered by events) are independent.  Calls that OVERLAP on the GPU race on the
 *             array and give wrong results: serialise them, or give the others a workspace of their own.
 *   Set-up    the array's device address is looked up once per device (cudaGetSymbolAddress, with that
 *             device current) on the first call there; umi_static_init() does only that, for callers who
 *             want it done before a capture or a timed loop starts.  `stream` must belong to the current device.
 * umi_static_scratch_bytes() returns UMI_STATIC_SCRATCH_BYTES (host only).
 */
#define UMI_STATIC_SCRATCH_BYTES (16u << 20)
size_t umi_static_scratch_bytes(void);
int umi_static_init(void);
int umi_detrend_gapped_static(const double* time, const float* flux,
                              int64_t n_stars, int64_t n_samples,
                              double t0, double dt, int64_t n_grid,
                              int W, float alpha, float c, int n_iter, int min_valid,
                              int64_t break_slots, int64_t min_segment, int64_t edge_cut,
                              float* trend_out, float* flat_out, void* stream);

/*
 * Batch driver (the paper streams 50-star batches): the same
 * computation with HOST buffers.  Stars are cut into batches of
 * `stars_per_batch` (<= 0: a body of ~32 MiB batches between a ramp up and a
 * ramp down by factors of 4, so that the first host->device copy and the last
 * device->host copy -- the only two no kernel hides -- are small), and
 * host->device copy, kernels and device->host copy of successive batches are
 * pipelined over `n_streams` CUDA streams (<= 0: 3, at most 16) with one device
 * buffer per stream.  Stream and buffer form a slot; slots are kept per device in a
 * free list between calls (the buffer is grown with cudaFree + cudaMalloc when a call
 * needs more; creating streams and allocating per call cost 0.3-0.5 ms of an 8 ms job),
 * taken when the call starts, given back when it returns, and freed by umi_shutdown().
 * Concurrent calls from several host threads are safe (each gets slots of its own).
 *
 *   time, flux, trend_out   HOST pointers, same shapes as above; time may be NULL.
 * The call returns after every batch has been copied back (it synchronises).
 */
int umi_detrend_host(const double* time, const float* flux,
                     int64_t n_stars, int64_t n_cadences,
                     int W, float alpha, int n_iter,
                     float* trend_out,
                     int64_t stars_per_batch, int n_streams);

/*
 * The batch driver with the normalisation fused in (detrending + normalization on a
 * whole sector from host memory): umi_detrend_host with c / min_valid exposed and
 * flat_out = flux / trend copied back as well.
 *   trend_out  HOST, float [n_stars*n_cadences], or NULL when only the flattened curve is wanted
 *              (the trend then never crosses PCIe).
 *   flat_out   HOST, float [n_stars*n_cadences]; required.
 * Everything else as umi_detrend_host.
 */
int umi_flatten_host(const double* time, const float* flux,
                     int64_t n_stars, int64_t n_cadences,
                     int W, float alpha, float c, int n_iter, int min_valid,
                     float* trend_out, float* flat_out,
                     int64_t stars_per_batch, int n_streams);

/*
 * Measurement aid: umi_detrend_ex, plus the device time of each of its two
 * kernels taken with CUDA events recorded on `stream` around each launch.
 *   kernel_ms  HOST, float[2]: [0] Phase-1 median kernel, [1] Phase-2/3
 *              reweighting kernel (0 when n_iter == 0), milliseconds.  Windows of
 *              at most 49 samples run all phases in one fused kernel: its time is
 *              reported in [1] and [0] is ~0.
 * Unlike umi_detrend this call SYNCHRONISES `stream` before returning.
 */
int umi_detrend_profile(const double* time, const float* flux,
                        int64_t n_stars, int64_t n_cadences,
                        int W, float alpha, float c, int n_iter, int min_valid,
                        float* trend_out, void* stream, float* kernel_ms);

/*
 * Launch geometry the library uses for this W (for reports and roofline
 * arithmetic; host only).  Any pointer may be NULL.
 *   median_tile    positions per CTA of the Phase-1 (median) kernel
 *   median_sort_n  power-of-two length of the per-tile sort
 *   weight_tile    positions per WARP tile of the Phase-2/3 (reweighting) kernel in its throughput variant
 *                  (batches of at most 4 CTAs of four such tiles per SM run the split-window variant: 1/8 of it)
 * Returns UMI_OK, or INVALID_ARG / UNSUPPORTED for a bad W.
 */
int umi_launch_geometry(int W, int* median_tile, int* median_sort_n, int* weight_tile);

/*
 * Releases what the HOST batch driver keeps between calls (its idle slots: streams and
 * device buffers, on every device it was used on).  Call it when no umi_*_host call is running;
 * the library can be used again afterwards.  Returns UMI_OK, or UMI_ERR_CUDA if a
 * destroy call failed.  The device entry points keep nothing, so programs that only use
 * those never need it.
 */
int umi_shutdown(void);

/* Static, never-freed string for a umi_status value. */
const char* umi_status_string(int status);

/* Library version: major*10000 + minor*100 + patch. */
int umi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* UMI_B200_H */
