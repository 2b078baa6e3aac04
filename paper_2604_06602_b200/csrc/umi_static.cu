/*
 * umi_static.cu -- umi_detrend_gapped_static (include/umi.h): the gap-handling path (R20, R23)
 * for callers that cannot allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
 *
 * umi_detrend_gapped[_ex] needs scratch memory (the slot grids its scatter, detrend and gather kernels pass to one another)
 * and takes it from the caller as a workspace.  Here the same kernels get it from a file-scope __device__ array of
 * UMI_STATIC_SCRATCH_BYTES that is part of the library's image: every GPU that loads the library holds it until the process
 * exits, nothing is allocated or freed by any call, and nothing about the existing entry points changes.
 *
 * In host code the array's NAME is a host-side stand-in for the symbol, not a device address.  The device address comes from
 * cudaGetSymbolAddress, asked once per device with that device current (below), and that pointer is what the kernels get.
 *
 * Every call on a device shares the one array, which keeps the previous call's contents: the path clears what it needs
 * (cudaMemsetAsync of the flux grid to the invalid pattern, first thing on the stream; every other region is written in full
 * before it is read), so calls that follow one another on a stream are independent -- but two calls that overlap on the GPU
 * (different streams, or different host threads without ordering between them) race on it.
 */
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

#include "umi.h"

/* 256-byte aligned: the carve-up into fp32 grids, 8-byte scan records and bytes keeps every region's natural alignment */
static __device__ __align__(256) unsigned char umi_static_scratch[UMI_STATIC_SCRATCH_BYTES];

namespace {

constexpr int MAX_DEVICES = 64;
std::mutex g_lock;
void* g_scratch[MAX_DEVICES];                               /* device address of the array, per device; null = not asked yet */

/* set-up, once per device, with that device current: the address of the array ON THE CURRENT DEVICE */
int scratch_address(void** out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return UMI_ERR_CUDA;
    }
    if (dev < 0 || dev >= MAX_DEVICES) return UMI_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> guard(g_lock);
    if (g_scratch[dev] == nullptr) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, umi_static_scratch);
        if (e != cudaSuccess || p == nullptr) {
            (void)cudaGetLastError();
            return UMI_ERR_CUDA;
        }
        g_scratch[dev] = p;
    }
    *out = g_scratch[dev];
    return UMI_OK;
}

} // namespace

extern "C" {

size_t umi_static_scratch_bytes(void) { return (size_t)UMI_STATIC_SCRATCH_BYTES; }

int umi_static_init(void)
{
    void* p = nullptr;
    return scratch_address(&p);
}

int umi_detrend_gapped_static(const double* time, const float* flux, int64_t n_stars, int64_t n_samples,
                              double t0, double dt, int64_t n_grid,
                              int W, float alpha, float c, int n_iter, int min_valid,
                              int64_t break_slots, int64_t min_segment, int64_t edge_cut,
                              float* trend_out, float* flat_out, void* stream)
{
    /* the size check comes first and needs no GPU: a job beyond the array is refused, never truncated */
    if (n_stars > 0 && n_grid > 0) {
        const bool segments = break_slots >= 0 || min_segment > 0 || edge_cut > 0;
        const size_t per_slot = segments ? 17 : 8;          /* umi_gapped_ex_workspace_bytes / umi_gapped_workspace_bytes */
        if ((uint64_t)n_stars > (uint64_t)UMI_STATIC_SCRATCH_BYTES / per_slot / (uint64_t)n_grid) return UMI_ERR_TOO_LARGE;
        const size_t need = segments ? umi_gapped_ex_workspace_bytes(n_stars, n_grid) : umi_gapped_workspace_bytes(n_stars, n_grid);
        if (need > (size_t)UMI_STATIC_SCRATCH_BYTES) return UMI_ERR_TOO_LARGE;
    }
    void* scratch = nullptr;
    const int st = scratch_address(&scratch);
    if (st != UMI_OK) return st;
    return umi_detrend_gapped_ex(time, flux, n_stars, n_samples, t0, dt, n_grid, W, alpha, c, n_iter, min_valid,
                                 break_slots, min_segment, edge_cut, trend_out, flat_out,
                                 scratch, (size_t)UMI_STATIC_SCRATCH_BYTES, stream);
}

} /* extern "C" */
