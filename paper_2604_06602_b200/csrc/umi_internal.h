/* umi_internal.h -- launch parameters shared by umi_kernels.cu and umi_api.cu (not installed). */
#ifndef UMI_INTERNAL_H
#define UMI_INTERNAL_H

#include <stdint.h>

namespace umi {

constexpr int K1_THREADS = 256;                  /* median kernel */
constexpr int K1_MIN_SORT = 1024;                /* smallest per-tile sort length */
constexpr int K1_BYTES_PER_SLOT = 14;            /* u64 sort entry + f32 median + u16 rank */

constexpr int K2_THREADS = 128;                  /* reweighting kernel */
constexpr int K2_NPOS = 4;                       /* consecutive positions per thread */
constexpr int K2_TILE = K2_THREADS * K2_NPOS;    /* positions per CTA */

struct MedianParams {
    const double* time;      /* may be null */
    const float* flux;
    float* out;              /* median, NaN where the position has no trend */
    int64_t N;               /* cadences per star */
    int64_t tiles_per_star;
    int64_t n_blocks;        /* n_stars * tiles_per_star */
    int W, T, NS, min_valid; /* T + W - 1 == NS */
};

struct ReweightParams {
    const double* time;
    const float* flux;
    float* out;              /* in: median from the median kernel; out: trend */
    int64_t N;
    int64_t tiles_per_star;
    int64_t n_blocks;
    int W, n_iter;
    float alpha, c;
};

__global__ void umi_median_kernel(MedianParams prm);
__global__ void umi_reweight_kernel(ReweightParams prm);

} // namespace umi

#endif
