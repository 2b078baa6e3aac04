/*
 * umi_regrid.cu -- gap handling by time stamps (the stage in front of the
 * detrender; reading R20).
 *
 * Mission pipelines deliver COMPACTED rows: cadences that failed quality filtering are
 * removed, so the time stamps jump.  The estimator of PAPER.md:35 is defined on W
 * consecutive cadence SLOTS (a fixed duration W*dt), so a compacted row is first put back
 * on its uniform grid:
 *     slot(b, i) = rint((time[b, i] - t0) / dt)            round half to even, fp64
 * scatter  grid_flux[b, slot] = flux[b, i]   (the grid is NaN-filled beforehand, so every
 *          gap becomes a run of invalid slots, which the detrender skips: R3)
 * detrend  the hot path on [n_stars, n_grid]
 * gather   trend_out[b, i] = grid_trend[b, slot],  flat_out[b, i] = flux[b, i] / trend.
 * A sample is invalid (NaN out, not scattered) iff its time or flux is not finite, its slot
 * falls outside [0, n_grid), or the NEXT sample of its row lands in the same slot (rows are
 * assumed non-decreasing in time; anything else is memory-safe but unspecified).
 *
 * Both kernels are pure data movement, four samples per thread with every load issued before its
 * first use, coalesced reads; the writes of the scatter and the reads of the gather are monotone
 * in the slot, i.e. coalesced except across gaps.  Bytes per sample: scatter 8 (time) + 4 (flux)
 * read, 4 written; gather 8 + 4 + 4 read, 4 (+4) written.  HBM-bound.
 * Nothing here is shared with oracle/.
 */
#include "umi_device.cuh"

namespace umi {

namespace {

constexpr int RG_THREADS = 256;

/* rint((t - t0)/dt) as a double (NaN-free input assumed finite), no range check */
__device__ __forceinline__ double raw_slot(double t, double t0, double dt)
{
    return rint(__ddiv_rn(__dsub_rn(t, t0), dt));     /* no contraction: same bits as the definition */
}

/*
 * Slot of a sample with the collision rule applied (flux not looked at), given its own time t (NaN
 * when the lane is outside the row).  One fp64 division per sample: the successor's slot comes from
 * the next lane by shuffle; only lane 31 computes it itself.  All 32 lanes must call this together.
 */
__device__ __forceinline__ int64_t sample_slot(double t, const double* __restrict__ trow, int64_t i, int64_t M,
                                               double t0, double dt, int64_t n_grid)
{
    const bool fin = finite_f64(t);
    const double k = fin ? raw_slot(t, t0, dt) : -1.0;
    double kn = __shfl_down_sync(0xFFFFFFFFu, k, 1);
    bool fin_n = __shfl_down_sync(0xFFFFFFFFu, (int)fin, 1) != 0;
    if ((threadIdx.x & 31) == 31) {
        fin_n = false;
        if (i + 1 < M) {
            const double tn = __ldg(trow + i + 1);
            fin_n = finite_f64(tn);
            if (fin_n) kn = raw_slot(tn, t0, dt);
        }
    }
    if (!fin || !(k >= 0.0) || !(k < (double)n_grid)) return -1;
    if (fin_n && kn == k) return -1;                    /* the next sample lands in the same slot */
    return (int64_t)k;
}

constexpr int RG_ITEMS = 4;                             /* samples per thread: all loads issued before any use */

/* grid = (chunks of a row, stars): no 64-bit division per sample */
__global__ void __launch_bounds__(RG_THREADS)
umi_regrid_scatter_kernel(RegridParams prm, float* __restrict__ grid_flux)
{
    const double dnan = __longlong_as_double(0x7FF8000000000000ll);
    for (int64_t b = blockIdx.y; b < prm.n_stars; b += gridDim.y) {
        const double* trow = prm.time + b * prm.M;
        const float* frow = prm.flux + b * prm.M;
        float* grow = grid_flux + b * prm.n_grid;
        for (int64_t base = (int64_t)blockIdx.x * (RG_THREADS * RG_ITEMS); base < prm.M;
             base += (int64_t)gridDim.x * (RG_THREADS * RG_ITEMS)) {
            double t[RG_ITEMS];
            float x[RG_ITEMS];
#pragma unroll
            for (int r = 0; r < RG_ITEMS; ++r) {
                const int64_t i = base + r * RG_THREADS + threadIdx.x;
                t[r] = i < prm.M ? __ldg(trow + i) : dnan;
                x[r] = i < prm.M ? __ldg(frow + i) : 0.f;
            }
#pragma unroll
            for (int r = 0; r < RG_ITEMS; ++r) {
                const int64_t i = base + r * RG_THREADS + threadIdx.x;
                const int64_t k = sample_slot(t[r], trow, i, prm.M, prm.t0, prm.dt, prm.n_grid);
                if (k >= 0 && finite_f32(x[r])) grow[k] = x[r];
            }
        }
    }
}

__global__ void __launch_bounds__(RG_THREADS)
umi_regrid_gather_kernel(RegridParams prm, const float* __restrict__ grid_trend, const uint8_t* __restrict__ grid_cut,
                         float* __restrict__ trend_out, float* __restrict__ flat_out)
{
    const float qnan = __int_as_float(0x7FC00000);
    const double dnan = __longlong_as_double(0x7FF8000000000000ll);
    for (int64_t b = blockIdx.y; b < prm.n_stars; b += gridDim.y) {
        const double* trow = prm.time + b * prm.M;
        const float* frow = prm.flux + b * prm.M;
        const float* grow = grid_trend + b * prm.n_grid;
        for (int64_t base = (int64_t)blockIdx.x * (RG_THREADS * RG_ITEMS); base < prm.M;
             base += (int64_t)gridDim.x * (RG_THREADS * RG_ITEMS)) {
            double t[RG_ITEMS];
            float x[RG_ITEMS], tr[RG_ITEMS];
#pragma unroll
            for (int r = 0; r < RG_ITEMS; ++r) {
                const int64_t i = base + r * RG_THREADS + threadIdx.x;
                t[r] = i < prm.M ? __ldg(trow + i) : dnan;
                x[r] = i < prm.M ? __ldg(frow + i) : 0.f;
            }
#pragma unroll
            for (int r = 0; r < RG_ITEMS; ++r) {
                const int64_t i = base + r * RG_THREADS + threadIdx.x;
                const int64_t k = sample_slot(t[r], trow, i, prm.M, prm.t0, prm.dt, prm.n_grid);
                tr[r] = (k >= 0 && finite_f32(x[r])) ? __ldg(grow + k) : qnan;
                if (grid_cut != nullptr && k >= 0 && __ldg(grid_cut + b * prm.n_grid + k)) tr[r] = qnan;   /* (R23) edge cut */
            }
#pragma unroll
            for (int r = 0; r < RG_ITEMS; ++r) {
                const int64_t i = base + r * RG_THREADS + threadIdx.x;
                if (i >= prm.M) continue;
                trend_out[b * prm.M + i] = tr[r];
                if (flat_out != nullptr) flat_out[b * prm.M + i] = (tr[r] == tr[r]) ? x[r] / tr[r] : qnan;
            }
        }
    }
}

/*
 * Segments (reading R23), on the slot grid after the scatter: the valid slots of a row are
 * cut into segments wherever more than break_slots empty slots lie between two of them; a segment with fewer
 * than min_segment valid slots is erased from grid_flux (NaN: in no window, no trend); grid_cut[k] = 1 for the
 * valid slots less than edge_cut slots from their segment's first or last slot (the gather blanks those).
 * One warp per row, 32 slots at a time, two passes: forward (first slot and index inside the segment, kept in
 * `scratch`), backward (last slot and size of the segment).  Windows need no clipping: the entry point only
 * accepts break_slots >= h, and a window of half-width h cannot reach across more than h - 1 empty slots.
 */
constexpr int SEG_BATCH = 8;                            /* chunks of 32 slots whose loads are issued together */

__global__ void __launch_bounds__(128)
umi_regrid_segments_kernel(float* __restrict__ grid_flux, uint8_t* __restrict__ grid_cut, int2* __restrict__ scratch,
                           int64_t n_stars, int64_t n_grid, int64_t break_slots, int64_t min_segment, int64_t edge_cut)
{
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u, le = lt | (1u << lane), gt = ~le;
    const float qnan = __int_as_float(0x7FC00000);
    for (int64_t b = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5); b < n_stars; b += (int64_t)gridDim.x * 4) {
        float* frow = grid_flux + b * n_grid;
        uint8_t* crow = grid_cut + b * n_grid;
        int2* srow = scratch + b * n_grid;
        /* forward: (first slot of the segment, index inside it) of every valid slot */
        bool have_prev = false;
        int64_t prev_slot = 0, cur_first = 0, cur_cnt = 0;
        for (int64_t base0 = 0; base0 < n_grid; base0 += 32 * SEG_BATCH) {
            bool vld[SEG_BATCH];                                    /* the chain between chunks is scalar: all loads of a batch first */
#pragma unroll
            for (int c = 0; c < SEG_BATCH; ++c) {
                const int64_t k = base0 + 32 * c + lane;
                vld[c] = k < n_grid && finite_f32(__ldcs(frow + k));
            }
#pragma unroll
            for (int c = 0; c < SEG_BATCH; ++c) {
                const int64_t base = base0 + 32 * c;
                if (base >= n_grid) break;
                const int64_t k = base + lane;
                const bool valid = vld[c];
                const unsigned vb = __ballot_sync(0xFFFFFFFFu, valid);
                const int p = 31 - __clz((int)(vb & lt));                           /* previous valid lane, -1: none */
                const bool none = p < 0 && !have_prev;
                const int64_t ps = p >= 0 ? base + p : prev_slot;
                const bool start = valid && (none || (break_slots >= 0 && k - ps - 1 > break_slots));
                const unsigned sb = __ballot_sync(0xFFFFFFFFu, start);
                if (valid) {
                    const int st = 31 - __clz((int)(sb & le));                      /* start lane of my segment, -1: before this chunk */
                    int2 rec;
                    if (st >= 0) { rec.x = (int)(base + st); rec.y = __popc(vb & le & ~((1u << st) - 1u)) - 1; }
                    else { rec.x = (int)cur_first; rec.y = (int)cur_cnt + __popc(vb & lt); }
                    srow[k] = rec;
                }
                if (vb) { prev_slot = base + 31 - __clz((int)vb); have_prev = true; }
                if (sb) { const int ls = 31 - __clz((int)sb); cur_first = base + ls; cur_cnt = __popc(vb & ~((1u << ls) - 1u)); }
                else cur_cnt += __popc(vb);
            }
        }
        __syncwarp();
        /* backward: (last slot, size) of the segment; short segments erased, edges marked */
        bool have_next = false;
        int64_t next_slot = 0, cur_last = 0, cur_total = 0;
        const int64_t top = ((n_grid - 1) / 32) * 32;
        for (int64_t base0 = top; base0 >= 0; base0 -= 32 * SEG_BATCH) {
            bool vld[SEG_BATCH];
            int2 recs[SEG_BATCH];
#pragma unroll
            for (int c = 0; c < SEG_BATCH; ++c) {
                const int64_t k = base0 - 32 * c + lane;
                vld[c] = k >= 0 && k < n_grid && finite_f32(frow[k]);
                recs[c] = vld[c] ? srow[k] : make_int2(0, 0);
            }
#pragma unroll
            for (int c = 0; c < SEG_BATCH; ++c) {
                const int64_t base = base0 - 32 * c;
                if (base < 0) break;
                const int64_t k = base + lane;
                const bool valid = vld[c];
                const int2 rec = recs[c];
                const unsigned vb = __ballot_sync(0xFFFFFFFFu, valid);
                const int nx = __ffs((int)(vb & gt)) - 1;                           /* next valid lane, -1: none */
                const bool none = nx < 0 && !have_next;
                const int64_t ns = nx >= 0 ? base + nx : next_slot;
                const bool end = valid && (none || (break_slots >= 0 && ns - k - 1 > break_slots));
                const unsigned eb = __ballot_sync(0xFFFFFFFFu, end);
                const int en = __ffs((int)(eb & ~lt)) - 1;                          /* end lane of my segment, -1: after this chunk */
                const int idx_at_end = __shfl_sync(0xFFFFFFFFu, rec.y, en >= 0 ? en : 0);
                const int64_t last = en >= 0 ? base + en : cur_last;
                const int64_t total = en >= 0 ? (int64_t)idx_at_end + 1 : cur_total;
                if (k < n_grid) {
                    const bool drop = valid && min_segment > 0 && total < min_segment;
                    if (drop) frow[k] = qnan;
                    crow[k] = (valid && !drop && edge_cut > 0 && (k - rec.x < edge_cut || last - k < edge_cut)) ? 1 : 0;
                }
                if (vb) { next_slot = base + __ffs((int)vb) - 1; have_next = true; }
                if (eb) {
                    const int fe = __ffs((int)eb) - 1;
                    cur_last = base + fe;
                    cur_total = (int64_t)__shfl_sync(0xFFFFFFFFu, rec.y, fe) + 1;
                }
            }
        }
    }
}

dim3 regrid_grid(int64_t n_stars, int64_t M)
{
    int64_t bx = (M + RG_THREADS * RG_ITEMS - 1) / (RG_THREADS * RG_ITEMS);
    if (bx < 1) bx = 1;
    if (bx > 1024) bx = 1024;
    int64_t by = n_stars < 1 ? 1 : n_stars;
    if (by > 65535) by = 65535;
    return dim3((unsigned)bx, (unsigned)by, 1);
}

} // namespace

cudaError_t launch_regrid_scatter(const RegridParams& prm, float* grid_flux, cudaStream_t stream)
{
    umi_regrid_scatter_kernel<<<regrid_grid(prm.n_stars, prm.M), RG_THREADS, 0, stream>>>(prm, grid_flux);
    return cudaGetLastError();
}

cudaError_t launch_regrid_gather(const RegridParams& prm, const float* grid_trend, const uint8_t* grid_cut, float* trend_out,
                                 float* flat_out, cudaStream_t stream)
{
    umi_regrid_gather_kernel<<<regrid_grid(prm.n_stars, prm.M), RG_THREADS, 0, stream>>>(prm, grid_trend, grid_cut,
                                                                                         trend_out, flat_out);
    return cudaGetLastError();
}

cudaError_t launch_regrid_segments(float* grid_flux, uint8_t* grid_cut, void* scratch, int64_t n_stars, int64_t n_grid,
                                   int64_t break_slots, int64_t min_segment, int64_t edge_cut, cudaStream_t stream)
{
    int64_t ctas = (n_stars + 3) / 4;
    if (ctas > 0x7FFFFFFF) ctas = 0x7FFFFFFF;
    umi_regrid_segments_kernel<<<(unsigned)ctas, 128, 0, stream>>>(grid_flux, grid_cut, static_cast<int2*>(scratch), n_stars,
                                                                    n_grid, break_slots, min_segment, edge_cut);
    return cudaGetLastError();
}

} // namespace umi
