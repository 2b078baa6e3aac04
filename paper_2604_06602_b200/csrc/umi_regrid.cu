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

/* rint((t - t0)/dt) as a double (NaN-free input assumed finite), no range check */
__device__ __forceinline__ double raw_slot(double t, double t0, double dt)
{
    return rint(__ddiv_rn(__dsub_rn(t, t0), dt));     /* no contraction: same bits as the definition */
}

/*
 * Slot of sample i of one row with the collision rule applied (flux not looked at).  One fp64
 * division per sample: the successor's slot comes from the next lane by shuffle; only lane 31
 * (and the last sample of a row) computes it itself.  All 32 lanes must call this together;
 * lanes with i >= M pass a NaN time and get -1.
 */
__device__ __forceinline__ int64_t sample_slot(const double* __restrict__ trow, int64_t i, int64_t M,
                                               double t0, double dt, int64_t n_grid)
{
    const bool in_row = i < M;
    const double t = in_row ? __ldg(trow + i) : __longlong_as_double(0x7FF8000000000000ll);
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

/* grid = (chunks of a row, stars): no 64-bit division per sample */
__global__ void __launch_bounds__(RG_THREADS)
umi_regrid_scatter_kernel(RegridParams prm, float* __restrict__ grid_flux)
{
    for (int64_t b = blockIdx.y; b < prm.n_stars; b += gridDim.y) {
        const double* trow = prm.time + b * prm.M;
        const float* frow = prm.flux + b * prm.M;
        float* grow = grid_flux + b * prm.n_grid;
        const int64_t Mr = (prm.M + 31) & ~(int64_t)31;             /* whole warps stay together */
        for (int64_t i = (int64_t)blockIdx.x * RG_THREADS + threadIdx.x; i < Mr; i += (int64_t)gridDim.x * RG_THREADS) {
            const int64_t k = sample_slot(trow, i, prm.M, prm.t0, prm.dt, prm.n_grid);
            if (k < 0) continue;
            const float x = __ldg(frow + i);
            if (finite_f32(x)) grow[k] = x;
        }
    }
}

__global__ void __launch_bounds__(RG_THREADS)
umi_regrid_gather_kernel(RegridParams prm, const float* __restrict__ grid_trend,
                         float* __restrict__ trend_out, float* __restrict__ flat_out)
{
    const float qnan = __int_as_float(0x7FC00000);
    for (int64_t b = blockIdx.y; b < prm.n_stars; b += gridDim.y) {
        const double* trow = prm.time + b * prm.M;
        const float* frow = prm.flux + b * prm.M;
        const float* grow = grid_trend + b * prm.n_grid;
        const int64_t Mr = (prm.M + 31) & ~(int64_t)31;
        for (int64_t i = (int64_t)blockIdx.x * RG_THREADS + threadIdx.x; i < Mr; i += (int64_t)gridDim.x * RG_THREADS) {
            const int64_t k = sample_slot(trow, i, prm.M, prm.t0, prm.dt, prm.n_grid);
            if (i >= prm.M) continue;
            const float x = __ldg(frow + i);
            float tr = qnan;
            if (k >= 0 && finite_f32(x)) tr = __ldg(grow + k);
            trend_out[b * prm.M + i] = tr;
            if (flat_out != nullptr) flat_out[b * prm.M + i] = (tr == tr) ? x / tr : qnan;
        }
    }
}

dim3 regrid_grid(int64_t n_stars, int64_t M)
{
    int64_t bx = (M + RG_THREADS - 1) / RG_THREADS;
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

cudaError_t launch_regrid_gather(const RegridParams& prm, const float* grid_trend, float* trend_out,
                                 float* flat_out, cudaStream_t stream)
{
    umi_regrid_gather_kernel<<<regrid_grid(prm.n_stars, prm.M), RG_THREADS, 0, stream>>>(prm, grid_trend,
                                                                                         trend_out, flat_out);
    return cudaGetLastError();
}

} // namespace umi
