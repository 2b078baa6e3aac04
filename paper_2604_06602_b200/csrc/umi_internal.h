/* umi_internal.h -- launch parameters and launch functions shared by the kernel files (umi_median.cu,
   umi_reweight.cu, umi_small.cu, umi_regrid.cu) and umi_api.cu (not installed). */
#ifndef UMI_INTERNAL_H
#define UMI_INTERNAL_H

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace umi {

#ifndef UMI_K1_THREADS
#define UMI_K1_THREADS 256
#endif
constexpr int K1_THREADS = UMI_K1_THREADS;       /* median kernel (128 for the 1024-key sort: launch_median) */
#ifndef UMI_K1_MIN_SORT
#define UMI_K1_MIN_SORT 1024
#endif
constexpr int K1_MIN_SORT = UMI_K1_MIN_SORT;     /* smallest per-tile sort length */
/* walkers per tile of the median kernel, per sort length, and its dynamic shared memory (bytes).  Measured:
   512 keys (small batches): one walker per position pair; 1024: three of the CTA's four warps; beyond that as many as
   leave the CTAs per SM of k1_min_ctas (umi_median.cu) their shared memory -- a multiple of 32, not necessarily a power of two.
   The MAD build stages one more fp32 per position: at 8192 keys it has room for 64 walkers only. */
#ifndef UMI_K1_WALKERS
#define UMI_K1_WALKERS(ns) ((ns) <= 512 ? 256 : 96)
#endif
__host__ __device__ constexpr int k1_walkers(int ns, bool mad = false)
{
    return (mad && ns >= 8192) ? 64 : ((mad && UMI_K1_WALKERS(ns) > 128) ? 128 : UMI_K1_WALKERS(ns));
}
/* t = positions per tile (T = ns - W + 1; 0: the worst case ns).  Layout: u64 sorted entries + u16 ranks + max(rank bitsets
   [NW][NS/32+1] + scan offsets [NW/32][NS/32], staging of the tile's results) + u32 sorted keys, one pad word per 32
   (k1_smem_base: the MAD build's scales start there) + in the MAD build one fp32 per position */
__host__ __device__ constexpr size_t k1_smem_base(int ns, bool mad, int t)
{
    const size_t bw = (size_t)ns / 32, nw = (size_t)k1_walkers(ns, mad);
    const size_t bits = 4 * (nw * (bw + 1) + (nw / 32) * bw);
    /* f32 medians [T], then u16 median ranks [T] and u16 window counts [T] (for n+ and the packed hand-over), rounded to 16 bytes */
    const size_t med = ((8 * (size_t)(t > 0 ? t : ns)) + 15) / 16 * 16;
    return (size_t)ns * 10 + (bits > med ? bits : med) + 4 * ((size_t)ns + (size_t)ns / 32);
}
__host__ __device__ constexpr size_t k1_smem_bytes(int ns, bool mad = false, int t = 0)
{
    return k1_smem_base(ns, mad, t) + (mad ? 4 * (size_t)ns : 0);
}

/* sibling estimators; values match include/umi.h */
constexpr int SCALE_UPPER_RMS = 0, SCALE_MAD = 1;
constexpr int WEIGHT_BISQUARE = 0, WEIGHT_WELSCH = 1;

constexpr int KS_THREADS = 128;                  /* fused small-window kernel: 4 consecutive positions per thread */
constexpr int KS_WARPS = KS_THREADS / 32;        /* every warp owns tiles of its own, as in the reweighting kernel */
constexpr int KS_WARP_TILE = 128;                /* positions per warp tile */
constexpr int KS_MAX_WINDOW = 49;                /* windows up to this length take the fused kernel */

#ifndef UMI_K2_THREADS
#define UMI_K2_THREADS 128
#endif
constexpr int K2_THREADS = UMI_K2_THREADS;       /* reweighting kernel */
constexpr int K2_WARPS = K2_THREADS / 32;        /* every warp owns tiles of its own: no CTA-wide barrier in the kernel */
constexpr int K2_NPOS = 4;                       /* consecutive positions per thread */
constexpr int K2_WARP_TILE = 32 * K2_NPOS;       /* positions per warp tile (throughput variant) */
#ifndef UMI_K2_SPLIT
#define UMI_K2_SPLIT 8
#endif
constexpr int K2_SPLIT = UMI_K2_SPLIT;                    /* small batches: lanes per 4 positions (warp tile = K2_WARP_TILE / K2_SPLIT) */

/* What the median kernel leaves in `out` for the reweighting kernel when passes follow (the paper's path):
   one 32-bit word per position, 0xFFFFFFFF = no trend here (R4, R5), else
       bits  0..15  offset of the median sample inside the window, 0 .. W-1 (the median IS a window sample)
       bits 16..31  n+ of Eq. 1 (R7), counted exactly on the sorted keys.
   The reweighting kernel has the window staged in shared memory and reads the median from there, so the
   two kernels need no scratch buffer besides `out` itself. */
constexpr uint32_t HANDOVER_NONE = 0xFFFFFFFFu;

struct MedianParams {
    const double* time;      /* may be null */
    const float* flux;
    float* out;              /* median, NaN where the position has no trend; or the packed hand-over words (above) */
    float* flat;             /* null, or flux / median (only set when the call stops after Phase 1) */
    float* scale;            /* null, or MAD of the window (selects the MAD variant of the kernel) */
    int packed;              /* 1: write the hand-over word (median offset | n+ << 16) instead of the median value */
    int64_t N;               /* cadences per star */
    int64_t tiles_per_star;
    int64_t n_blocks;        /* n_stars * tiles_per_star */
    int W, T, NS, min_valid; /* T + W - 1 == NS */
};

struct ReweightParams {
    const double* time;
    const float* flux;
    float* out;              /* in: from the median kernel (hand-over words if `packed`, else medians); out: trend */
    float* flat;             /* null, or flux / trend (PAPER.md:155 normalisation), NaN where trend is NaN */
    const float* scale_in;   /* family kernels: null, or s per position (replaces Phase 2) */
    float* scale_out;        /* family kernels: null, or receives s per position */
    int packed;              /* 1: `out` holds hand-over words (the paper's path), 0: fp32 medians (sibling estimators) */
    int split;               /* reweighting kernel: 1, or K2_SPLIT for batches too small to fill the GPU */
    int weight_kind;         /* family kernels: WEIGHT_BISQUARE / WEIGHT_WELSCH */
    int scale_kind;          /* fused short-window kernel only */
    int64_t N;
    int64_t tiles_per_star;  /* reweighting kernel: WARP tiles per star */
    int64_t n_blocks;        /* n_stars * tiles_per_star */
    int W, n_iter;
    float alpha, c;
    float c_over_alpha;      /* c / alpha, formed on the host: the sentinel's distance factor ("Sentinel") */
};

/* Enqueue one kernel; return the launch status (cudaGetLastError). */
cudaError_t launch_median(const MedianParams& prm, unsigned grid, size_t smem, cudaStream_t stream);
/* family = false: the paper's path (scale_in/scale_out/weight_kind ignored); true: the sibling-estimator variants */
cudaError_t launch_reweight(const ReweightParams& prm, bool family, unsigned grid, size_t smem, cudaStream_t stream);
/* fused kernel for W <= KS_MAX_WINDOW; wt = compiled wire count (9, 17, 25, 33 or 49) >= W; prm.tiles_per_star and
   prm.n_blocks count WARP tiles of KS_WARP_TILE positions, grid = CTAs of KS_WARPS warps */
cudaError_t launch_small(const ReweightParams& prm, bool family, int min_valid, int wt, unsigned grid, cudaStream_t stream);

/* umi_regrid.cu: gap handling by time stamps (R20) */
struct RegridParams {
    const double* time;      /* [n_stars, M] compacted rows */
    const float* flux;       /* [n_stars, M] */
    int64_t n_stars, M, n_grid;
    double t0, dt;
};
/* grid_flux[n_stars, n_grid] must already be NaN-filled */
cudaError_t launch_regrid_scatter(const RegridParams& prm, float* grid_flux, cudaStream_t stream);
/* trend_out[b, i] = grid_trend[b, slot] (NaN for invalid samples, and where grid_cut (nullable) marks the slot);
   flat_out (nullable) = flux / trend */
cudaError_t launch_regrid_gather(const RegridParams& prm, const float* grid_trend, const uint8_t* grid_cut, float* trend_out,
                                 float* flat_out, cudaStream_t stream);
/* segments on the slot grid (reading R23): erases short segments from grid_flux, marks edge slots in grid_cut
   [n_stars, n_grid]; scratch: 8 bytes per slot */
cudaError_t launch_regrid_segments(float* grid_flux, uint8_t* grid_cut, void* scratch, int64_t n_stars, int64_t n_grid,
                                   int64_t break_slots, int64_t min_segment, int64_t edge_cut, cudaStream_t stream);

} // namespace umi

#endif
