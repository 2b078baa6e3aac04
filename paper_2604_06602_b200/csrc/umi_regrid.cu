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

/*
 * The same with one CTA of SEGP_WARPS warps per row, for batches with too few rows to fill the GPU with one warp each
 * (1,000 rows of 19,440 slots: 1,000 warps, each a chain of 608 dependent chunk steps, twice).  Warp p owns the p-th part of
 * the row's chunks.  What a part does to the scan state depends on the state it receives only through its FIRST valid
 * slot (does a segment start there?); everything else -- its last valid slot, its count, the last segment start strictly
 * inside it -- is the part's own.  So: a summary pass per part, the summaries folded in order (at most SEGP_WARPS - 1 steps,
 * every warp for itself), then the scan proper with the right state coming in.  The backward pass needs no summary pass of its
 * own: a segment END strictly inside a part is the valid slot in front of a START strictly inside it, which the forward pass
 * has just seen.  Results are identical to umi_regrid_segments_kernel (same records, same flags).
 * Measured on config 2 (1,000 rows x 19,440 slots), whole F2-with-segments step over the base path: warp per row +0.72 ms;
 * 8 warps per row +0.55 (104 registers), 8 / 4 CTAs per SM +0.49, 16 / 2 +0.47 (batch 4: 64 registers, no spills; batch 8
 * spilled), 16 / 1 +0.54-0.57, 32 / 1 +0.53, 4 / 8 +0.51.
 */
#ifndef UMI_SEGP_WARPS
#define UMI_SEGP_WARPS 16
#endif
#ifndef UMI_SEGP_MIN_CTAS
#define UMI_SEGP_MIN_CTAS 2     /* 64 registers, nothing spilled with SEGP_BATCH = 4 */
#endif
constexpr int SEGP_WARPS = UMI_SEGP_WARPS;
#ifndef UMI_SEGP_BATCH
#define UMI_SEGP_BATCH 4
#endif
constexpr int SEGP_BATCH = UMI_SEGP_BATCH;          /* chunks whose loads are issued together */

struct SegPart {                /* forward summary of a part; slots are 32-bit (n_grid <= 2^31 - 1) */
    int fv, lv, nv;             /* first / last valid slot (-1: none), number of valid slots */
    int ls, cnt_ls;             /* last segment start strictly inside the part (-1: none), valid slots from it to the part's end */
    int e_low, tot_low;         /* backward: lowest segment end strictly inside the part (-1: none), size of the segment ending there */
    int idx_lv;                 /* backward: index inside its segment of the part's last valid slot */
};

__global__ void __launch_bounds__(32 * SEGP_WARPS, UMI_SEGP_MIN_CTAS)
umi_regrid_segments_cta_kernel(float* __restrict__ grid_flux, uint8_t* __restrict__ grid_cut, int2* __restrict__ scratch,
                               int64_t n_stars, int64_t n_grid, int64_t break_slots, int64_t min_segment, int64_t edge_cut)
{
    __shared__ SegPart part[SEGP_WARPS];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt = (1u << lane) - 1u, le = lt | (1u << lane), gt = ~le;
    const float qnan = __int_as_float(0x7FC00000);
    const int64_t n_chunks = (n_grid + 31) / 32;
    const int64_t cpp = (n_chunks + SEGP_WARPS - 1) / SEGP_WARPS;          /* chunks per part */
    const int64_t c_lo = warp * cpp, c_hi = (c_lo + cpp < n_chunks) ? c_lo + cpp : n_chunks;   /* my chunks [c_lo, c_hi) */
    for (int64_t b = blockIdx.x; b < n_stars; b += gridDim.x) {
        float* frow = grid_flux + b * n_grid;
        uint8_t* crow = grid_cut + b * n_grid;
        int2* srow = scratch + b * n_grid;
        /* 1. summary of my part (valid bits only; starts strictly inside: both slots of the gap are mine) */
        {
            int fv = -1, lv = -1, nv = 0, ls = -1, cnt_ls = 0;
            for (int64_t c0 = c_lo; c0 < c_hi; c0 += SEGP_BATCH) {
                bool vld[SEGP_BATCH];
#pragma unroll
                for (int c = 0; c < SEGP_BATCH; ++c) {
                    const int64_t k = (c0 + c) * 32 + lane;
                    vld[c] = c0 + c < c_hi && k < n_grid && finite_f32(__ldcg(frow + k));
                }
#pragma unroll
                for (int c = 0; c < SEGP_BATCH; ++c) {
                    if (c0 + c >= c_hi) break;
                    const int base = (int)((c0 + c) * 32);
                    const unsigned vb = __ballot_sync(0xFFFFFFFFu, vld[c]);
                    if (vb == 0u) continue;
                    const int p = 31 - __clz((int)(vb & lt));
                    const int ps = p >= 0 ? base + p : lv;                          /* previous valid slot inside the part, -1: none */
                    const bool start = vld[c] && ps >= 0 && break_slots >= 0 && (int64_t)(base + lane) - ps - 1 > break_slots;
                    const unsigned sb = __ballot_sync(0xFFFFFFFFu, start);
                    if (fv < 0) fv = base + __ffs((int)vb) - 1;
                    lv = base + 31 - __clz((int)vb);
                    nv += __popc(vb);
                    if (sb) { const int l2 = 31 - __clz((int)sb); ls = base + l2; cnt_ls = __popc(vb & ~((1u << l2) - 1u)); }
                    else cnt_ls += __popc(vb);
                }
            }
            if (lane == 0) { part[warp].fv = fv; part[warp].lv = lv; part[warp].nv = nv; part[warp].ls = ls; part[warp].cnt_ls = cnt_ls; }
        }
        __syncthreads();
        /* 2. the state my part receives: parts 0 .. warp-1 folded in order */
        bool have_prev = false;
        int64_t prev_slot = 0, cur_first = 0, cur_cnt = 0;
        for (int q = 0; q < warp; ++q) {
            const SegPart s = part[q];
            if (s.nv == 0) continue;
            const bool bstart = !have_prev || (break_slots >= 0 && (int64_t)s.fv - prev_slot - 1 > break_slots);
            if (s.ls >= 0) { cur_first = s.ls; cur_cnt = s.cnt_ls; }
            else if (bstart) { cur_first = s.fv; cur_cnt = s.nv; }
            else cur_cnt += s.nv;
            prev_slot = s.lv;
            have_prev = true;
        }
        /* 3. forward over my part: (first slot of the segment, index inside it) of every valid slot; on the way, the lowest
              segment end strictly inside the part (the valid slot in front of the first start strictly inside it) */
        {
            int e_low = -1, tot_low = 0, idx_lv = 0;
            int own_prev = -1, own_prev_idx = 0;                                    /* my part's previous valid slot and its index */
            for (int64_t c0 = c_lo; c0 < c_hi; c0 += SEGP_BATCH) {
                bool vld[SEGP_BATCH];
#pragma unroll
                for (int c = 0; c < SEGP_BATCH; ++c) {
                    const int64_t k = (c0 + c) * 32 + lane;
                    vld[c] = c0 + c < c_hi && k < n_grid && finite_f32(__ldcg(frow + k));
                }
#pragma unroll
                for (int c = 0; c < SEGP_BATCH; ++c) {
                    if (c0 + c >= c_hi) break;
                    const int64_t base = (c0 + c) * 32;
                    const int64_t k = base + lane;
                    const bool valid = vld[c];
                    const unsigned vb = __ballot_sync(0xFFFFFFFFu, valid);
                    const int p = 31 - __clz((int)(vb & lt));
                    const bool none = p < 0 && !have_prev;
                    const int64_t ps = p >= 0 ? base + p : prev_slot;
                    const bool start = valid && (none || (break_slots >= 0 && k - ps - 1 > break_slots));
                    const unsigned sb = __ballot_sync(0xFFFFFFFFu, start);
                    int my_idx = 0;
                    if (valid) {
                        const int st = 31 - __clz((int)(sb & le));
                        int2 rec;
                        if (st >= 0) { rec.x = (int)(base + st); rec.y = __popc(vb & le & ~((1u << st) - 1u)) - 1; }
                        else { rec.x = (int)cur_first; rec.y = (int)cur_cnt + __popc(vb & lt); }
                        srow[k] = rec;
                        my_idx = rec.y;
                    }
                    if (vb) {
                        /* the first start strictly inside the part: its previous valid slot is mine (own_prev, or a lane of this chunk) */
                        if (e_low < 0 && sb) {
                            unsigned cand = sb;
                            if (own_prev < 0) cand &= ~(1u << (__ffs((int)vb) - 1));     /* the part's very first valid slot: its predecessor is not mine */
                            if (cand) {
                                const int sl = __ffs((int)cand) - 1;                /* lane of that start */
                                const unsigned below = vb & ((1u << sl) - 1u);
                                if (below) {
                                    const int pl = 31 - __clz((int)below);
                                    e_low = (int)base + pl;
                                    tot_low = __shfl_sync(0xFFFFFFFFu, my_idx, pl) + 1;
                                } else {
                                    e_low = own_prev;
                                    tot_low = own_prev_idx + 1;
                                }
                            }
                        }
                        const int hl = 31 - __clz((int)vb);
                        own_prev = (int)base + hl;
                        own_prev_idx = __shfl_sync(0xFFFFFFFFu, my_idx, hl);
                        idx_lv = own_prev_idx;
                        prev_slot = base + hl;
                        have_prev = true;
                    }
                    if (sb) { const int l2 = 31 - __clz((int)sb); cur_first = base + l2; cur_cnt = __popc(vb & ~((1u << l2) - 1u)); }
                    else cur_cnt += __popc(vb);
                }
            }
            if (lane == 0) { part[warp].e_low = e_low; part[warp].tot_low = tot_low; part[warp].idx_lv = idx_lv; }
        }
        __syncthreads();                                            /* records and summaries are complete */
        /* 4. the state my part receives going backward: parts SEGP_WARPS-1 .. warp+1 folded in order */
        bool have_next = false;
        int64_t next_slot = 0, cur_last = 0, cur_total = 0;
        for (int q = SEGP_WARPS - 1; q > warp; --q) {
            const SegPart s = part[q];
            if (s.nv == 0) continue;
            const bool bend = !have_next || (break_slots >= 0 && next_slot - (int64_t)s.lv - 1 > break_slots);
            if (s.e_low >= 0) { cur_last = s.e_low; cur_total = s.tot_low; }
            else if (bend) { cur_last = s.lv; cur_total = (int64_t)s.idx_lv + 1; }
            next_slot = s.fv;
            have_next = true;
        }
        /* 5. backward over my part: (last slot, size) of the segment; short segments erased, edges marked */
        for (int64_t c0 = c_hi - 1; c0 >= c_lo; c0 -= SEGP_BATCH) {
            bool vld[SEGP_BATCH];
            int2 recs[SEGP_BATCH];
#pragma unroll
            for (int c = 0; c < SEGP_BATCH; ++c) {
                const int64_t k = (c0 - c) * 32 + lane;
                vld[c] = c0 - c >= c_lo && k < n_grid && finite_f32(frow[k]);
                recs[c] = vld[c] ? srow[k] : make_int2(0, 0);
            }
#pragma unroll
            for (int c = 0; c < SEGP_BATCH; ++c) {
                if (c0 - c < c_lo) break;
                const int64_t base = (c0 - c) * 32;
                const int64_t k = base + lane;
                const bool valid = vld[c];
                const int2 rec = recs[c];
                const unsigned vb = __ballot_sync(0xFFFFFFFFu, valid);
                const int nx = __ffs((int)(vb & gt)) - 1;
                const bool none = nx < 0 && !have_next;
                const int64_t ns = nx >= 0 ? base + nx : next_slot;
                const bool end = valid && (none || (break_slots >= 0 && ns - k - 1 > break_slots));
                const unsigned eb = __ballot_sync(0xFFFFFFFFu, end);
                const int en = __ffs((int)(eb & ~lt)) - 1;
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
        __syncthreads();                                            /* part[] is free for the next row */
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
    /* rows enough to fill the GPU with a warp each (64 warps x ~150 SMs): one warp per row; fewer: a CTA per row */
#ifndef UMI_SEG_CTA_BELOW
#define UMI_SEG_CTA_BELOW 4096
#endif
    if (n_stars < UMI_SEG_CTA_BELOW) {
        umi_regrid_segments_cta_kernel<<<(unsigned)n_stars, 32 * SEGP_WARPS, 0, stream>>>(grid_flux, grid_cut, static_cast<int2*>(scratch),
                                                                                            n_stars, n_grid, break_slots, min_segment, edge_cut);
        return cudaGetLastError();
    }
    int64_t ctas = (n_stars + 3) / 4;
    if (ctas > 0x7FFFFFFF) ctas = 0x7FFFFFFF;
    umi_regrid_segments_kernel<<<(unsigned)ctas, 128, 0, stream>>>(grid_flux, grid_cut, static_cast<int2*>(scratch), n_stars,
                                                                    n_grid, break_slots, min_segment, edge_cut);
    return cudaGetLastError();
}

} // namespace umi
