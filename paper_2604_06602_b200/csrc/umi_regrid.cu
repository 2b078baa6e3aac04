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
 * Both kernels are pure data movement, one thread per sample, coalesced reads; the writes
 * of the scatter and the reads of the gather are monotone in the slot, i.e. coalesced
 * except across gaps.  Bytes per sample: scatter 8 (time) + 4 (flux) + 8 (next time, L1/L2
 * hit) read, 4 written; gather 8 + 4 + 4 read, 4 (+4) written.  HBM-bound.
 * Nothing here is shared with oracle/.
 */
#include "umi_device.cuh"

namespace umi {

namespace {

constexpr int RG_THREADS = 256;

/* slot of a time stamp, or -1 */
__device__ __forceinline__ int64_t slot_of(double t, double t0, double dt, int64_t n_grid)
{
    if (!finite_f64(t)) return -1;
    const double k = rint(__ddiv_rn(__dsub_rn(t, t0), dt));   /* no contraction: same bits as the definition */
    if (!(k >= 0.0) || !(k < (double)n_grid)) return -1;
    return (int64_t)k;
}

/* slot of sample (row, i) with the collision rule applied (flux not looked at) */
__device__ __forceinline__ int64_t sample_slot(const double* __restrict__ trow, int64_t i, int64_t M,
                                               double t0, double dt, int64_t n_grid)
{
    const int64_t k = slot_of(__ldg(trow + i), t0, dt, n_grid);
    if (k < 0) return -1;
    if (i + 1 < M) {
        const double tn = __ldg(trow + i + 1);
        if (finite_f64(tn) && rint(__ddiv_rn(__dsub_rn(tn, t0), dt)) == (double)k) return -1;
    }
    return k;
}

__global__ void __launch_bounds__(RG_THREADS)
umi_regrid_scatter_kernel(RegridParams prm, float* __restrict__ grid_flux)
{
    const int64_t total = prm.n_stars * prm.M;
    for (int64_t q = (int64_t)blockIdx.x * RG_THREADS + threadIdx.x; q < total;
         q += (int64_t)gridDim.x * RG_THREADS) {
        const int64_t b = q / prm.M, i = q - b * prm.M;
        const int64_t k = sample_slot(prm.time + b * prm.M, i, prm.M, prm.t0, prm.dt, prm.n_grid);
        if (k < 0) continue;
        const float x = __ldg(prm.flux + q);
        if (finite_f32(x)) grid_flux[b * prm.n_grid + k] = x;
    }
}

__global__ void __launch_bounds__(RG_THREADS)
umi_regrid_gather_kernel(RegridParams prm, const float* __restrict__ grid_trend,
                         float* __restrict__ trend_out, float* __restrict__ flat_out)
{
    const int64_t total = prm.n_stars * prm.M;
    const float qnan = __int_as_float(0x7FC00000);
    for (int64_t q = (int64_t)blockIdx.x * RG_THREADS + threadIdx.x; q < total;
         q += (int64_t)gridDim.x * RG_THREADS) {
        const int64_t b = q / prm.M, i = q - b * prm.M;
        const int64_t k = sample_slot(prm.time + b * prm.M, i, prm.M, prm.t0, prm.dt, prm.n_grid);
        const float x = __ldg(prm.flux + q);
        float tr = qnan;
        if (k >= 0 && finite_f32(x)) tr = __ldg(grid_trend + b * prm.n_grid + k);
        trend_out[q] = tr;
        if (flat_out != nullptr) flat_out[q] = (tr == tr) ? x / tr : qnan;
    }
}

unsigned regrid_grid(int64_t total)
{
    int64_t blocks = (total + RG_THREADS - 1) / RG_THREADS;
    const int64_t cap = 148 * 16;                       /* grid-stride: 16 CTAs of 256 per SM */
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    return (unsigned)blocks;
}

} // namespace

cudaError_t launch_regrid_scatter(const RegridParams& prm, float* grid_flux, cudaStream_t stream)
{
    umi_regrid_scatter_kernel<<<regrid_grid(prm.n_stars * prm.M), RG_THREADS, 0, stream>>>(prm, grid_flux);
    return cudaGetLastError();
}

cudaError_t launch_regrid_gather(const RegridParams& prm, const float* grid_trend, float* trend_out,
                                 float* flat_out, cudaStream_t stream)
{
    umi_regrid_gather_kernel<<<regrid_grid(prm.n_stars * prm.M), RG_THREADS, 0, stream>>>(prm, grid_trend,
                                                                                         trend_out, flat_out);
    return cudaGetLastError();
}

} // namespace umi
