/*
 * umi_api.cu -- the C ABI of include/umi.h: argument validation, launch
 * geometry, kernel launches and the host-buffer batch driver.
 */
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#include <algorithm>
#include <mutex>
#include <vector>

#include "umi.h"
#include "umi_internal.h"

namespace {

constexpr int64_t MAX_GRID = 0x7FFFFFFF;

/* sibling-estimator selection (F4); the default is the paper's path */
struct Family {
    bool on = false;
    int scale_kind = umi::SCALE_UPPER_RMS, weight_kind = umi::WEIGHT_BISQUARE;
    float* scale_out = nullptr;
};

struct Geometry {
    int T1, NS;            /* median kernel: positions per tile, sort length */
    size_t smem1;
    int halo4;             /* reweighting kernel: staged floats per warp besides its tile (4 per float4 group) */
};

/* DESIGN.md, "Launch geometry": the sort length is the smallest power of two
   (>= 1024) that leaves at least (W-1)/2 positions per tile. */
Geometry geometry_for(int W)
{
    Geometry g;
    int ns = umi::K1_MIN_SORT;
    while (ns < (W - 1) + (W - 1) / 2) ns <<= 1;
    g.NS = ns;
    g.T1 = ns - (W - 1);
    g.smem1 = umi::k1_smem_bytes(ns, false, g.T1);
    const int h = (W - 1) / 2;
    const int hal = (h + 3) & ~3;
    const int G = (3 + (hal - h) + 2 * h) / 4 + 1;
    g.halo4 = 4 * G;
    return g;
}

/* SMs of the current device (sizes the "does this batch fill the GPU" decision); 148 on B200 */
int sm_count()
{
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
        (void)cudaGetLastError();
        return 148;
    }
    return n;
}

int check_window(int W)
{
    if (W < 1 || (W & 1) == 0) return UMI_ERR_INVALID_ARG;
    if (W > UMI_MAX_WINDOW) return UMI_ERR_UNSUPPORTED;
    return UMI_OK;
}

int cuda_failed(cudaError_t e)
{
    if (e == cudaSuccess) return 0;
    (void)cudaGetLastError(); /* clear */
    return 1;
}

int validate(const float* flux, int64_t n_stars, int64_t n_cadences, int W, float alpha, float c,
             int n_iter, const float* trend_out)
{
    if (flux == nullptr || trend_out == nullptr) return UMI_ERR_INVALID_ARG;
    if (n_stars < 0 || n_cadences < 0 || n_iter < 0) return UMI_ERR_INVALID_ARG;
    if (!(alpha > 0.f) || !isfinite(alpha) || !(c > 0.f) || !isfinite(c)) return UMI_ERR_INVALID_ARG;
    return check_window(W);
}

/* Enqueue the kernels of one call for device-resident buffers.  Allocates nothing: the only scratch the two
   kernels share is trend_out itself (umi_internal.h, "hand-over word"). */
int launch_device(const double* time, const float* flux, int64_t n_stars, int64_t n_cadences,
                  int W, float alpha, float c, int n_iter, int min_valid, float* trend_out,
                  cudaStream_t stream, cudaEvent_t* ev = nullptr /* [3] or null */,
                  float* flat_out = nullptr, const Family& fam = Family(),
                  bool in_pipeline = false /* other batches keep the GPU busy: pick the throughput variants whatever the size */)
{
    if (n_stars == 0 || n_cadences == 0) return UMI_OK;
    Geometry g = geometry_for(W);
    const bool mad = fam.on && fam.scale_kind == umi::SCALE_MAD;
    /* small batches (fewer median tiles than SMs; config 1 has 30): a 512-key sort with tiles of at least 128
       positions gives four times the CTAs and a shorter serial chain in each (latency is what is left to win) */
    if (!in_pipeline && W - 1 + 128 <= 512 && n_stars * ((n_cadences + g.T1 - 1) / g.T1) < (int64_t)sm_count()) {   /* (forced on the large batches it loses: config 5 8.9 vs 7.3 ms per 20,000 stars, config 2 1.27 vs 0.63 ms) */
        g.NS = 512;
        g.T1 = 512 - (W - 1);
        g.smem1 = umi::k1_smem_bytes(g.NS, false, g.T1);
    }
    if (mad) g.smem1 = umi::k1_smem_bytes(g.NS, true, g.T1);
    if (min_valid < 0) min_valid = std::max(1, W / 3);      /* PAPER.md:192 (R4) */

    if (W <= umi::KS_MAX_WINDOW) {
        /* short windows: all three phases in one register-resident kernel (umi_small.cu) */
        umi::ReweightParams rp;
        rp.time = time;
        rp.flux = flux;
        rp.out = trend_out;
        rp.flat = flat_out;
        rp.N = n_cadences;
        rp.tiles_per_star = (n_cadences + umi::KS_WARP_TILE - 1) / umi::KS_WARP_TILE;
        rp.n_blocks = n_stars * rp.tiles_per_star;
        rp.W = W;
        rp.n_iter = n_iter;
        rp.alpha = alpha;
        rp.c = c;
        rp.c_over_alpha = c / alpha;
        rp.split = 1;
        rp.packed = 0;
        rp.scale_in = nullptr;
        rp.scale_out = fam.scale_out;
        rp.weight_kind = fam.weight_kind;
        rp.scale_kind = fam.scale_kind;
        const int wt = W <= 9 ? 9 : W <= 17 ? 17 : W <= 25 ? 25 : W <= 33 ? 33 : 49;
        const unsigned grid = (unsigned)std::min<int64_t>((rp.n_blocks + umi::KS_WARPS - 1) / umi::KS_WARPS, MAX_GRID);
        if (ev && (cuda_failed(cudaEventRecord(ev[0], stream)) || cuda_failed(cudaEventRecord(ev[1], stream))))
            return UMI_ERR_CUDA;
        if (cuda_failed(umi::launch_small(rp, fam.on, min_valid, wt, grid, stream))) return UMI_ERR_CUDA;
        if (ev && cuda_failed(cudaEventRecord(ev[2], stream))) return UMI_ERR_CUDA;
        return UMI_OK;
    }

    /* the family path also runs the second kernel with n_iter = 0 when only the upper-RMS scale is wanted */
    const bool scale_only = fam.on && !mad && fam.scale_out != nullptr && n_iter == 0;
    const bool second = n_iter > 0 || scale_only;
    /* The paper's path with passes to run: the median kernel leaves, per position, where in its window the
       median sample sits and n+ (Eq. 1's count, exact on the sorted keys) in trend_out; the reweighting
       kernel reads both back and overwrites them with the trend. */
    const int packed = (!fam.on && n_iter > 0) ? 1 : 0;

    umi::MedianParams mp;
    mp.time = time;
    mp.flux = flux;
    mp.out = trend_out;
    mp.flat = second ? nullptr : flat_out;                  /* whichever kernel writes the final trend divides */
    mp.scale = mad ? fam.scale_out : nullptr;
    mp.packed = packed;
    mp.N = n_cadences;
    mp.tiles_per_star = (n_cadences + g.T1 - 1) / g.T1;
    mp.n_blocks = n_stars * mp.tiles_per_star;
    mp.W = W;
    mp.T = g.T1;
    mp.NS = g.NS;
    mp.min_valid = min_valid;
    const unsigned grid1 = (unsigned)std::min<int64_t>(mp.n_blocks, MAX_GRID);
    if (ev && cuda_failed(cudaEventRecord(ev[0], stream))) return UMI_ERR_CUDA;
    if (cuda_failed(umi::launch_median(mp, grid1, g.smem1, stream))) return UMI_ERR_CUDA;
    if (ev && cuda_failed(cudaEventRecord(ev[1], stream))) return UMI_ERR_CUDA;

    if (second) {
        umi::ReweightParams rp;
        rp.time = time;
        rp.flux = flux;
        rp.out = trend_out;
        rp.flat = flat_out;
        rp.N = n_cadences;
        rp.split = 1;
        rp.packed = packed;
        int wtile = umi::K2_WARP_TILE;
        rp.tiles_per_star = (n_cadences + wtile - 1) / wtile;
        rp.n_blocks = n_stars * rp.tiles_per_star;
        if (!fam.on && !in_pipeline && (rp.n_blocks + umi::K2_WARPS - 1) / umi::K2_WARPS <= 4 * (int64_t)sm_count()) {
            /* the grid would leave most of the resident-CTA slots empty: split every window over
               K2_SPLIT lanes instead (latency, not throughput, is what is left to win) */
            rp.split = umi::K2_SPLIT;
            wtile = umi::K2_WARP_TILE / umi::K2_SPLIT;
            rp.tiles_per_star = (n_cadences + wtile - 1) / wtile;
            rp.n_blocks = n_stars * rp.tiles_per_star;
        }
        rp.W = W;
        rp.n_iter = n_iter;
        rp.alpha = alpha;
        rp.c = c;
        rp.c_over_alpha = c / alpha;
        rp.scale_in = mad ? fam.scale_out : nullptr;
        rp.scale_out = mad ? nullptr : fam.scale_out;
        rp.weight_kind = fam.weight_kind;
        rp.scale_kind = fam.scale_kind;
        const unsigned grid2 = (unsigned)std::min<int64_t>((rp.n_blocks + umi::K2_WARPS - 1) / umi::K2_WARPS, MAX_GRID);
        const size_t smem2 = (size_t)umi::K2_WARPS * (size_t)(wtile + g.halo4) * sizeof(float);
        if (cuda_failed(umi::launch_reweight(rp, fam.on, grid2, smem2, stream))) return UMI_ERR_CUDA;
    }
    if (ev && cuda_failed(cudaEventRecord(ev[2], stream))) return UMI_ERR_CUDA;
    return UMI_OK;
}

} // namespace

extern "C" {

int umi_window_len(double dt_days)
{
    if (!(dt_days > 0.0) || !isfinite(dt_days)) return 0;
    const double q = (0.5 / dt_days) * (1.0 + 1.0 / 1048576.0);     /* (R15) */
    if (!(q < 2147483646.0)) return 0;
    return (int)floor(q) | 1;
}

int umi_detrend_ex(const double* time, const float* flux, int64_t n_stars, int64_t n_cadences,
                   int W, float alpha, float c, int n_iter, int min_valid,
                   float* trend_out, void* stream)
{
    const int st = validate(flux, n_stars, n_cadences, W, alpha, c, n_iter, trend_out);
    if (st != UMI_OK) return st;
    return launch_device(time, flux, n_stars, n_cadences, W, alpha, c, n_iter, min_valid, trend_out,
                         static_cast<cudaStream_t>(stream));
}

int umi_flatten(const double* time, const float* flux, int64_t n_stars, int64_t n_cadences,
                int W, float alpha, float c, int n_iter, int min_valid,
                float* trend_out, float* flat_out, void* stream)
{
    if (flat_out == nullptr) return UMI_ERR_INVALID_ARG;
    const int st = validate(flux, n_stars, n_cadences, W, alpha, c, n_iter, trend_out);
    if (st != UMI_OK) return st;
    return launch_device(time, flux, n_stars, n_cadences, W, alpha, c, n_iter, min_valid, trend_out,
                         static_cast<cudaStream_t>(stream), nullptr, flat_out);
}

int umi_detrend_family(const double* time, const float* flux, int64_t n_stars, int64_t n_cadences,
                       int W, int scale_kind, int weight_kind, float alpha, float c, int n_iter, int min_valid,
                       float* trend_out, float* scale_out, float* flat_out, void* stream)
{
    if (scale_kind != UMI_SCALE_UPPER_RMS && scale_kind != UMI_SCALE_MAD) return UMI_ERR_INVALID_ARG;
    if (weight_kind != UMI_WEIGHT_BISQUARE && weight_kind != UMI_WEIGHT_WELSCH) return UMI_ERR_INVALID_ARG;
    if (scale_kind == UMI_SCALE_MAD && scale_out == nullptr) return UMI_ERR_INVALID_ARG;
    const int st = validate(flux, n_stars, n_cadences, W, alpha, c, n_iter, trend_out);
    if (st != UMI_OK) return st;
    Family fam;
    fam.on = true;
    fam.scale_kind = scale_kind;
    fam.weight_kind = weight_kind;
    fam.scale_out = scale_out;
    return launch_device(time, flux, n_stars, n_cadences, W, alpha, c, n_iter, min_valid, trend_out,
                         static_cast<cudaStream_t>(stream), nullptr, flat_out, fam);
}

size_t umi_gapped_workspace_bytes(int64_t n_stars, int64_t n_grid)
{
    if (n_stars <= 0 || n_grid <= 0) return 0;
    /* two fp32 grids: flux on the slots, and the trend on the slots */
    return (size_t)n_stars * (size_t)n_grid * (2 * sizeof(float));
}

size_t umi_gapped_ex_workspace_bytes(int64_t n_stars, int64_t n_grid)
{
    if (n_stars <= 0 || n_grid <= 0) return 0;
    /* the two grids, 8 bytes per slot for the segment scan, one edge-cut byte per slot */
    return (size_t)n_stars * (size_t)n_grid * (2 * sizeof(float) + 2 * sizeof(int32_t) + 1);
}

int umi_detrend_gapped_ex(const double* time, const float* flux, int64_t n_stars, int64_t n_samples,
                          double t0, double dt, int64_t n_grid,
                          int W, float alpha, float c, int n_iter, int min_valid,
                          int64_t break_slots, int64_t min_segment, int64_t edge_cut,
                          float* trend_out, float* flat_out,
                          void* workspace, size_t workspace_bytes, void* stream)
{
    if (time == nullptr || n_grid < 0 || !(dt > 0.0) || !isfinite(dt) || !isfinite(t0)) return UMI_ERR_INVALID_ARG;
    const int st = validate(flux, n_stars, n_samples, W, alpha, c, n_iter, trend_out);
    if (st != UMI_OK) return st;
    if (n_grid > 0x7FFFFFFF) return UMI_ERR_UNSUPPORTED;              /* slots are 32-bit in the segment scan */
    const bool segments = break_slots >= 0 || min_segment > 0 || edge_cut > 0;
    /* windows are never clipped at a break: a break the window could reach across is refused (umi.h) */
    if (break_slots >= 0 && break_slots < (W - 1) / 2) return UMI_ERR_UNSUPPORTED;
    if (n_stars == 0 || n_samples == 0) return UMI_OK;
    const size_t need = segments ? umi_gapped_ex_workspace_bytes(n_stars, n_grid) : umi_gapped_workspace_bytes(n_stars, n_grid);
    if (need > 0 && (workspace == nullptr || workspace_bytes < need)) return UMI_ERR_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    umi::RegridParams gp;
    gp.time = time;
    gp.flux = flux;
    gp.n_stars = n_stars;
    gp.M = n_samples;
    gp.n_grid = n_grid;
    gp.t0 = t0;
    gp.dt = dt;
    const size_t slots = (size_t)n_stars * (size_t)n_grid;
    float* grid_flux = static_cast<float*>(workspace);
    float* grid_trend = grid_flux + slots;
    void* scan = grid_trend + slots;                                  /* 8 bytes per slot, 8-byte aligned */
    uint8_t* grid_cut = segments ? static_cast<uint8_t*>(scan) + slots * 8 : nullptr;
    if (n_grid > 0) {
        /* 0xFFFFFFFF is a NaN: every slot starts invalid */
        if (cuda_failed(cudaMemsetAsync(grid_flux, 0xFF, slots * sizeof(float), s))) return UMI_ERR_CUDA;
        if (cuda_failed(umi::launch_regrid_scatter(gp, grid_flux, s))) return UMI_ERR_CUDA;
        if (segments && cuda_failed(umi::launch_regrid_segments(grid_flux, grid_cut, scan, n_stars, n_grid, break_slots,
                                                                min_segment, edge_cut, s)))
            return UMI_ERR_CUDA;
        const int st2 = launch_device(nullptr, grid_flux, n_stars, n_grid, W, alpha, c, n_iter, min_valid,
                                      grid_trend, s);
        if (st2 != UMI_OK) return st2;
    }
    if (cuda_failed(umi::launch_regrid_gather(gp, grid_trend, n_grid > 0 ? grid_cut : nullptr, trend_out, flat_out, s)))
        return UMI_ERR_CUDA;
    return UMI_OK;
}

int umi_detrend_gapped(const double* time, const float* flux, int64_t n_stars, int64_t n_samples,
                       double t0, double dt, int64_t n_grid,
                       int W, float alpha, float c, int n_iter, int min_valid,
                       float* trend_out, float* flat_out,
                       void* workspace, size_t workspace_bytes, void* stream)
{
    return umi_detrend_gapped_ex(time, flux, n_stars, n_samples, t0, dt, n_grid, W, alpha, c, n_iter, min_valid,
                                 -1, 0, 0, trend_out, flat_out, workspace, workspace_bytes, stream);
}

int umi_detrend_profile(const double* time, const float* flux, int64_t n_stars, int64_t n_cadences,
                        int W, float alpha, float c, int n_iter, int min_valid,
                        float* trend_out, void* stream, float* kernel_ms)
{
    if (kernel_ms == nullptr) return UMI_ERR_INVALID_ARG;
    kernel_ms[0] = kernel_ms[1] = 0.f;
    int st = validate(flux, n_stars, n_cadences, W, alpha, c, n_iter, trend_out);
    if (st != UMI_OK) return st;
    if (n_stars == 0 || n_cadences == 0) return UMI_OK;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    for (auto& e : ev)
        if (cuda_failed(cudaEventCreate(&e))) st = UMI_ERR_CUDA;
    if (st == UMI_OK)
        st = launch_device(time, flux, n_stars, n_cadences, W, alpha, c, n_iter, min_valid, trend_out, s, ev);
    if (st == UMI_OK && cuda_failed(cudaEventSynchronize(ev[2]))) st = UMI_ERR_CUDA;
    if (st == UMI_OK &&
        (cuda_failed(cudaEventElapsedTime(&kernel_ms[0], ev[0], ev[1])) ||
         cuda_failed(cudaEventElapsedTime(&kernel_ms[1], ev[1], ev[2]))))
        st = UMI_ERR_CUDA;
    for (auto& e : ev)
        if (e) (void)cudaEventDestroy(e);
    return st;
}

int umi_detrend(const double* time, const float* flux, int64_t n_stars, int64_t n_cadences,
                int W, float alpha, int n_iter, float* trend_out, void* stream)
{
    return umi_detrend_ex(time, flux, n_stars, n_cadences, W, alpha, 5.0f /* PAPER.md:63 */, n_iter, -1,
                          trend_out, stream);
}

} /* extern "C" */

namespace {

/* What the HOST batch driver keeps between calls, per device: a free list of SLOTS, each a CUDA stream and one device
   buffer that is only ever grown (creating and destroying three streams per call cost ~0.3 ms of an 8.7 ms config-2 job;
   allocating the buffers per call another 0.1-0.2 ms).  A call takes the slots it needs under the mutex and puts them back
   when it returns, so concurrent callers never share a stream or a buffer; umi_shutdown() frees everything.  No memory
   pool, of the device or of the library, is involved.  The DEVICE entry points use none of this. */
constexpr int MAX_DEVICES = 64;
struct DriverSlot {
    cudaStream_t stream = nullptr;
    void* buf = nullptr;
    size_t cap = 0;
};
struct HostDriverState {
    std::mutex lock;
    std::vector<DriverSlot> idle[MAX_DEVICES];
};
HostDriverState& driver_state()
{
    static HostDriverState* st = new HostDriverState();     /* never destroyed: no CUDA call from a static destructor */
    return *st;
}

/* n slots of the current device, each with a buffer of at least `bytes` (grown with cudaFree + cudaMalloc when it is not) */
bool take_slots(int dev, int n, size_t bytes, std::vector<DriverSlot>& out)
{
    out.clear();
    if (dev < 0 || dev >= MAX_DEVICES) return false;
    HostDriverState& st = driver_state();
    {
        std::lock_guard<std::mutex> guard(st.lock);
        while ((int)out.size() < n && !st.idle[dev].empty()) {
            out.push_back(st.idle[dev].back());
            st.idle[dev].pop_back();
        }
    }
    while ((int)out.size() < n) {
        DriverSlot s;
        if (cuda_failed(cudaStreamCreateWithFlags(&s.stream, cudaStreamNonBlocking))) return false;
        out.push_back(s);
    }
    for (auto& s : out) {
        if (s.cap >= bytes) continue;
        if (s.buf != nullptr) (void)cudaFree(s.buf);
        s.buf = nullptr;
        s.cap = 0;
        if (cuda_failed(cudaMalloc(&s.buf, bytes))) return false;
        s.cap = bytes;
    }
    return true;
}

void return_slots(int dev, std::vector<DriverSlot>& slots)
{
    if (dev < 0 || dev >= MAX_DEVICES) return;
    HostDriverState& st = driver_state();
    std::lock_guard<std::mutex> guard(st.lock);
    for (const DriverSlot& s : slots) st.idle[dev].push_back(s);
    slots.clear();
}

/* the batch driver behind umi_detrend_host / umi_flatten_host: trend_out and flat_out are HOST pointers,
   either may be null (not both) */
int host_driver(const double* time, const float* flux, int64_t n_stars, int64_t n_cadences,
                int W, float alpha, float c, int n_iter, int min_valid, float* trend_out, float* flat_out,
                int64_t stars_per_batch, int n_streams)
{
    if (trend_out == nullptr && flat_out == nullptr) return UMI_ERR_INVALID_ARG;
    const int st = validate(flux, n_stars, n_cadences, W, alpha, c, n_iter, trend_out ? trend_out : flat_out);
    if (st != UMI_OK) return st;
    if (n_stars == 0 || n_cadences == 0) return UMI_OK;
    if (n_streams <= 0) n_streams = 3;
    if (n_streams > 16) n_streams = 16;
    /* batch sizes.  Given by the caller: uniform.  Default: a body of ~32 MiB batches between a ramp up and
       a ramp down by factors of 4 (body/64, body/16, body/4, body ..., body/4, body/16, body/64): only the
       first host->device copy and the last device->host copy are not hidden behind a kernel, so those two
       batches are made small, and a factor of 4 keeps every copy shorter than the kernels it runs beside
       (the kernels take ~6x longer per star than one copy at W = 361 and PCIe 5 x16). */
    std::vector<int64_t> sizes;
    if (stars_per_batch > 0) {
        stars_per_batch = std::min(stars_per_batch, n_stars);
        for (int64_t left = n_stars; left > 0; left -= std::min(stars_per_batch, left))
            sizes.push_back(std::min(stars_per_batch, left));
    } else {
        const int64_t row_bytes = std::max<int64_t>(n_cadences * (int64_t)sizeof(float), 1);
        int64_t body = std::max<int64_t>(1, (32ll << 20) / row_bytes);
        body = std::min(body, std::max<int64_t>(1, (n_stars * 3) / 5));     /* ramps take ~2/3 of a body */
        const int64_t ramp[3] = {std::max<int64_t>(1, body / 64), std::max<int64_t>(1, body / 16),
                                 std::max<int64_t>(1, body / 4)};
        int64_t left = n_stars;
        for (int i = 0; i < 3 && left > 0 && ramp[i] < body; ++i) {
            sizes.push_back(std::min(ramp[i], left));
            left -= sizes.back();
        }
        const int64_t tail = ramp[0] + ramp[1] + ramp[2];
        while (left > tail) {
            sizes.push_back(std::min(body, left - tail));
            left -= sizes.back();
        }
        for (int i = 2; i >= 0 && left > 0; --i) {
            sizes.push_back(std::min(ramp[i], left));
            left -= sizes.back();
        }
        if (left > 0) sizes.push_back(left);
        stars_per_batch = *std::max_element(sizes.begin(), sizes.end());
    }
    const int64_t n_batches = (int64_t)sizes.size();
    if ((int64_t)n_streams > n_batches) n_streams = (int)n_batches;

    struct Slot {
        cudaStream_t stream = nullptr;
        float* d_flux = nullptr;
        float* d_trend = nullptr;
        float* d_flat = nullptr;
        double* d_time = nullptr;
    };
    std::vector<Slot> slots((size_t)n_streams);
    const size_t elems = (size_t)stars_per_batch * (size_t)n_cadences;
    int status = UMI_OK;

    /* one cached buffer per slot, carved into time | flux | trend | flat (each region a multiple of 256 bytes) */
    auto region = [](size_t bytes) { return (bytes + 255) / 256 * 256; };
    const size_t b_time = time != nullptr ? region(elems * sizeof(double)) : 0;
    const size_t b_f32 = region(elems * sizeof(float));
    const size_t b_slot = b_time + b_f32 * (flat_out != nullptr ? 3 : 2);
    int dev = 0;
    if (cuda_failed(cudaGetDevice(&dev))) return UMI_ERR_CUDA;
    std::vector<DriverSlot> held;
    if (!take_slots(dev, n_streams, b_slot, held)) {
        return_slots(dev, held);
        return UMI_ERR_CUDA;
    }
    for (size_t i = 0; i < slots.size(); ++i) {
        unsigned char* base = static_cast<unsigned char*>(held[i].buf);
        slots[i].stream = held[i].stream;
        slots[i].d_time = time != nullptr ? reinterpret_cast<double*>(base) : nullptr;
        slots[i].d_flux = reinterpret_cast<float*>(base + b_time);
        slots[i].d_trend = reinterpret_cast<float*>(base + b_time + b_f32);
        slots[i].d_flat = flat_out != nullptr ? reinterpret_cast<float*>(base + b_time + 2 * b_f32) : nullptr;
    }

    int64_t s0 = 0;
    for (int64_t b = 0; status == UMI_OK && b < n_batches; s0 += sizes[(size_t)b], ++b) {
        Slot& s = slots[(size_t)(b % n_streams)];
        const int64_t ns = sizes[(size_t)b];
        const size_t off = (size_t)s0 * (size_t)n_cadences;
        const size_t cnt = (size_t)ns * (size_t)n_cadences;
        /* the slot's stream serialises reuse of its buffers */
        if (cuda_failed(cudaMemcpyAsync(s.d_flux, flux + off, cnt * sizeof(float), cudaMemcpyHostToDevice, s.stream)) ||
            (time != nullptr &&
             cuda_failed(cudaMemcpyAsync(s.d_time, time + off, cnt * sizeof(double), cudaMemcpyHostToDevice, s.stream)))) {
            status = UMI_ERR_CUDA;
            break;
        }
        /* a batch between other batches is not alone on the GPU: its small-batch (latency) variants would only cost issue
           slots the neighbours could use (config 2 end to end: 7.84 -> see DESIGN.md section 7) */
        status = launch_device(s.d_time, s.d_flux, ns, n_cadences, W, alpha, c, n_iter, min_valid, s.d_trend, s.stream,
                               nullptr, s.d_flat, Family(), n_batches > 1);
        if (status != UMI_OK) break;
        if ((trend_out != nullptr &&
             cuda_failed(cudaMemcpyAsync(trend_out + off, s.d_trend, cnt * sizeof(float), cudaMemcpyDeviceToHost, s.stream))) ||
            (flat_out != nullptr &&
             cuda_failed(cudaMemcpyAsync(flat_out + off, s.d_flat, cnt * sizeof(float), cudaMemcpyDeviceToHost, s.stream))))
            status = UMI_ERR_CUDA;
    }

    for (auto& s : slots)
        if (s.stream != nullptr && cuda_failed(cudaStreamSynchronize(s.stream))) status = UMI_ERR_CUDA;
    (void)cudaGetLastError();
    return_slots(dev, held);
    return status;
}

} // namespace

extern "C" {

int umi_shutdown(void)
{
    HostDriverState& st = driver_state();
    std::lock_guard<std::mutex> guard(st.lock);
    int status = UMI_OK;
    bool any = false;
    for (int dev = 0; dev < MAX_DEVICES; ++dev) any = any || !st.idle[dev].empty();
    if (!any) return UMI_OK;                                /* nothing kept: no CUDA call at all */
    int before = 0;
    const bool have_dev = cudaGetDevice(&before) == cudaSuccess;
    for (int dev = 0; dev < MAX_DEVICES; ++dev) {
        if (st.idle[dev].empty()) continue;
        if (cuda_failed(cudaSetDevice(dev))) { status = UMI_ERR_CUDA; continue; }
        for (const DriverSlot& s : st.idle[dev]) {
            if (s.buf != nullptr && cuda_failed(cudaFree(s.buf))) status = UMI_ERR_CUDA;
            if (s.stream != nullptr && cuda_failed(cudaStreamDestroy(s.stream))) status = UMI_ERR_CUDA;
        }
        st.idle[dev].clear();
    }
    if (have_dev) (void)cudaSetDevice(before);
    (void)cudaGetLastError();
    return status;
}

int umi_detrend_host(const double* time, const float* flux, int64_t n_stars, int64_t n_cadences,
                     int W, float alpha, int n_iter, float* trend_out,
                     int64_t stars_per_batch, int n_streams)
{
    if (trend_out == nullptr) return UMI_ERR_INVALID_ARG;
    return host_driver(time, flux, n_stars, n_cadences, W, alpha, 5.0f /* PAPER.md:63 */, n_iter, -1, trend_out, nullptr,
                       stars_per_batch, n_streams);
}

int umi_flatten_host(const double* time, const float* flux, int64_t n_stars, int64_t n_cadences,
                     int W, float alpha, float c, int n_iter, int min_valid,
                     float* trend_out, float* flat_out, int64_t stars_per_batch, int n_streams)
{
    if (flat_out == nullptr) return UMI_ERR_INVALID_ARG;
    return host_driver(time, flux, n_stars, n_cadences, W, alpha, c, n_iter, min_valid, trend_out, flat_out,
                       stars_per_batch, n_streams);
}

int umi_launch_geometry(int W, int* median_tile, int* median_sort_n, int* weight_tile)
{
    const int st = check_window(W);
    if (st != UMI_OK) return st;
    const Geometry g = geometry_for(W);
    if (median_tile) *median_tile = g.T1;
    if (median_sort_n) *median_sort_n = g.NS;
    if (weight_tile) *weight_tile = umi::K2_WARP_TILE;
    return UMI_OK;
}

const char* umi_status_string(int status)
{
    switch (status) {
    case UMI_OK: return "UMI_OK";
    case UMI_ERR_INVALID_ARG: return "UMI_ERR_INVALID_ARG: null pointer, negative size, even or < 1 window, or bad alpha/c/n_iter";
    case UMI_ERR_UNSUPPORTED: return "UMI_ERR_UNSUPPORTED: window longer than UMI_MAX_WINDOW";
    case UMI_ERR_CUDA: return "UMI_ERR_CUDA: a CUDA launch, copy or allocation failed";
    case UMI_ERR_TOO_LARGE: return "UMI_ERR_TOO_LARGE: the job needs more scratch than the static array of UMI_STATIC_SCRATCH_BYTES holds";
    default: return "UMI: unknown status";
    }
}

int umi_version(void) { return 400; /* 0.4.0: umi_detrend_gapped_static, UMI_ERR_TOO_LARGE */ }

} /* extern "C" */
