/*
 * umi_bakeoff.cu -- the ALTERNATIVES that were measured against the product kernels (not product:
 * built into libumi_bakeoff.so by `python -m paper_2604_06602_b200.build --bakeoff`, run by
 * `python -m paper_2604_06602_b200.bakeoff`; results in profiles/ and DESIGN.md section 6).
 *
 * Phase 1, the two selection schemes north_star names beside the product's
 * "sort the tile once + sliding walkers" (umi_median.cu):
 *   (i)  umi_bakeoff_median_radix        shared-memory radix select: a warp per position, the W keys of
 *                                        the window in registers, 4 passes over 8-bit digits with a
 *                                        per-warp shared-memory histogram; exact.
 *   (ii) umi_bakeoff_median_warp_sorted  an incrementally maintained sorted window per warp: the window's
 *                                        keys sorted across the 32 lanes (K consecutive ranks per lane); a
 *                                        slide deletes the leaving key and inserts the entering one by
 *                                        shifting registers (one shuffle at each lane boundary); exact.
 * Phases 2-3, the mapping north_star names beside the product's "thread owns 4
 * positions, no reductions" (umi_reweight.cu):
 *   (iii) umi_bakeoff_reweight_warp_window  a warp per window, its samples in registers (ceil(W/32) per
 *                                        lane), the sums of Eq. 1 and Eq. 4 by xor shuffles; same packed
 *                                        arithmetic as the product kernel (umi_device.cuh).
 * And the prior art itself, for scale:
 *   (0)  umi_bakeoff_paper_design        the paper's kernel design: one thread per (star, position)
 *                                        copies its window into a private array (local memory), finds the median by
 *                                        quickselect, then one upper-RMS pass and n_iter reweighting passes over the array;
 *                                        written from that description, fp32, same readings (R1-R18).
 * Same validity rules as the product path (R2-R6, R16): NaN out where the own sample is invalid or the
 * window holds fewer than min_valid valid samples; lower middle for even counts.  No `time` argument.
 */
#include <cuda_runtime.h>
#include <stdint.h>

#include "umi_device.cuh"

namespace {

using namespace umi;

constexpr int BK_THREADS = 256;
constexpr int BK_WARPS = BK_THREADS / 32;
constexpr int BK_TILE = 256;                     /* positions per CTA (selection (i), mapping (iii)) */
constexpr int64_t BK_MAX_GRID = 0x7FFFFFFF;

/* ------------------------------------------------------------------ (i) radix select, warp per position */
template <int KPL>
__global__ void __launch_bounds__(BK_THREADS)
bk_median_radix(const float* __restrict__ flux, int64_t N, int64_t tiles_per_star, int64_t n_blocks, int W, int min_valid,
                float* __restrict__ out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint32_t* keys = reinterpret_cast<uint32_t*>(smem_raw);         /* [BK_TILE + W - 1] */
    uint32_t* hist = keys + ((BK_TILE + W - 1 + 3) & ~3);           /* [BK_WARPS][256] */
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int h = (W - 1) >> 1;
    uint32_t* myhist = hist + warp * 256;
    for (int64_t bid = blockIdx.x; bid < n_blocks; bid += gridDim.x) {
        const int64_t star = bid / tiles_per_star, tile = bid - star * tiles_per_star;
        const int64_t j0 = tile * BK_TILE;
        const float* frow = flux + star * N;
        for (int u = tid; u < BK_TILE + W - 1; u += BK_THREADS) {
            float x = 0.f;
            const bool ok = load_sample(nullptr, frow, N, j0 - h + u, x);
            keys[u] = ok ? float_to_key(x) : KEY_INVALID;
        }
        __syncthreads();
        for (int p = warp; p < BK_TILE && j0 + p < N; p += BK_WARPS) {
            uint32_t k[KPL];
            int n = 0;
#pragma unroll
            for (int i = 0; i < KPL; ++i) {
                const int o = lane + 32 * i;
                k[i] = (o < W) ? keys[p + o] : KEY_INVALID;
                n += (k[i] != KEY_INVALID) ? 1 : 0;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xFFFFFFFFu, n, o);
            const bool own = keys[p + h] != KEY_INVALID;
            float res = __int_as_float(0x7FC00000);
            if (own && n >= min_valid && n > 0) {
                int target = (n - 1) >> 1;                          /* (R6) */
                uint32_t prefix = 0u, mask = 0u;
#pragma unroll 1
                for (int shift = 24; shift >= 0; shift -= 8) {
#pragma unroll
                    for (int b = 0; b < 8; ++b) myhist[lane * 8 + b] = 0u;
                    __syncwarp();
#pragma unroll
                    for (int i = 0; i < KPL; ++i)
                        if (k[i] != KEY_INVALID && (k[i] & mask) == prefix) atomicAdd(&myhist[(k[i] >> shift) & 255u], 1u);
                    __syncwarp();
                    /* lane owns bins 8*lane .. 8*lane+7; exclusive prefix over lanes, then the bin holding `target` */
                    uint32_t c[8];
                    int mine = 0;
#pragma unroll
                    for (int b = 0; b < 8; ++b) { c[b] = myhist[lane * 8 + b]; mine += (int)c[b]; }
                    int incl = mine;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int t = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                        if (lane >= o) incl += t;
                    }
                    int cum = incl - mine;
                    int bin = -1, before = 0;
#pragma unroll
                    for (int b = 0; b < 8; ++b) {
                        if (bin < 0 && target < cum + (int)c[b]) { bin = lane * 8 + b; before = cum; }
                        cum += (int)c[b];
                    }
                    const unsigned who = __ballot_sync(0xFFFFFFFFu, bin >= 0);
                    const int src = __ffs((int)who) - 1;
                    bin = __shfl_sync(0xFFFFFFFFu, bin, src);
                    before = __shfl_sync(0xFFFFFFFFu, before, src);
                    target -= before;
                    prefix |= (uint32_t)bin << shift;
                    mask |= 255u << shift;
                    __syncwarp();
                }
                res = key_to_float(prefix);
            }
            if (lane == 0) out[star * N + j0 + p] = res;
        }
        __syncthreads();
    }
}

/* ------------------------------------------------------------------ (ii) sorted window maintained per warp */
template <int K>
struct SortedWindow {
    uint32_t e[K];                                                  /* global sorted index = lane*K + j; unused slots = KEY_INVALID */
    __device__ __forceinline__ void clear()
    {
#pragma unroll
        for (int j = 0; j < K; ++j) e[j] = KEY_INVALID;
    }
    /* number of stored keys strictly below `key` = index of its first occurrence / its insertion point */
    __device__ __forceinline__ int lower_bound(uint32_t key) const
    {
        int c = 0;
#pragma unroll
        for (int j = 0; j < K; ++j) c += (e[j] < key) ? 1 : 0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xFFFFFFFFu, c, o);
        return c;
    }
    __device__ __forceinline__ void insert(uint32_t key, int lane)
    {
        const int pos = lower_bound(key);
        const uint32_t carry = __shfl_up_sync(0xFFFFFFFFu, e[K - 1], 1);
        const int base = lane * K;
#pragma unroll
        for (int j = K - 1; j >= 1; --j) {
            const int gi = base + j;
            e[j] = gi > pos ? e[j - 1] : (gi == pos ? key : e[j]);
        }
        e[0] = base > pos ? carry : (base == pos ? key : e[0]);
    }
    __device__ __forceinline__ void remove(uint32_t key, int lane)
    {
        const int pos = lower_bound(key);
        uint32_t carry = __shfl_down_sync(0xFFFFFFFFu, e[0], 1);
        if (lane == 31) carry = KEY_INVALID;
        const int base = lane * K;
#pragma unroll
        for (int j = 0; j < K - 1; ++j) e[j] = (base + j >= pos) ? e[j + 1] : e[j];
        e[K - 1] = (base + K - 1 >= pos) ? carry : e[K - 1];
    }
    __device__ __forceinline__ uint32_t at(int r, int lane) const
    {
        const int j = r % K;
        uint32_t v = e[0];
#pragma unroll
        for (int jj = 1; jj < K; ++jj) v = (j == jj) ? e[jj] : v;
        return __shfl_sync(0xFFFFFFFFu, v, r / K);
    }
};

template <int K>
__global__ void __launch_bounds__(128)
bk_median_warp_sorted(const float* __restrict__ flux, int64_t N, int64_t runs_per_star, int64_t n_runs, int run, int W, int min_valid,
                      float* __restrict__ out)
{
    const int lane = threadIdx.x & 31;
    const int h = (W - 1) >> 1;
    const float qnan = __int_as_float(0x7FC00000);
    for (int64_t rid = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5); rid < n_runs; rid += (int64_t)gridDim.x * 4) {
        const int64_t star = rid / runs_per_star, r0 = rid - star * runs_per_star;
        const int64_t p0 = r0 * run;
        const int64_t p1 = (p0 + run < N) ? p0 + run : N;
        const float* frow = flux + star * N;
        SortedWindow<K> win;
        win.clear();
        int n = 0;
        /* first window [p0 - h, p0 + h]: one insertion per valid sample (amortised over the run) */
        for (int64_t j = p0 - h; j <= p0 + h; ++j) {
            float x = 0.f;
            if (load_sample(nullptr, frow, N, j, x)) { win.insert(float_to_key(x), lane); ++n; }   /* (uniform: every lane reads the same j) */
        }
        for (int64_t p = p0; p < p1; ++p) {
            float own = 0.f;
            const bool own_ok = load_sample(nullptr, frow, N, p, own);
            float res = qnan;
            if (own_ok && n >= min_valid && n > 0) res = key_to_float(win.at((n - 1) >> 1, lane));
            if (lane == 0) out[star * N + p] = res;
            if (p + 1 < p1) {
                float xo = 0.f, xi = 0.f;
                if (load_sample(nullptr, frow, N, p - h, xo)) { win.remove(float_to_key(xo), lane); --n; }
                if (load_sample(nullptr, frow, N, p + 1 + h, xi)) { win.insert(float_to_key(xi), lane); ++n; }
            }
        }
    }
}

/* ------------------------------------------------------------------ (iii) Phases 2-3, a warp per window */
template <int KPL, int APOW>
__global__ void __launch_bounds__(BK_THREADS)
bk_reweight_warp_window(const float* __restrict__ flux, const float* __restrict__ median, int64_t N, int64_t tiles_per_star,
                        int64_t n_blocks, int W, float alpha, float c, int n_iter, float* __restrict__ out)
{
    static_assert(KPL % 2 == 0, "pairs");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* xs = reinterpret_cast<float*>(smem_raw);                 /* [BK_TILE + W - 1], NaN = invalid */
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int h = (W - 1) >> 1;
    const float qnan = __int_as_float(0x7FC00000);
    const float nalpha = -alpha;
    for (int64_t bid = blockIdx.x; bid < n_blocks; bid += gridDim.x) {
        const int64_t star = bid / tiles_per_star, tile = bid - star * tiles_per_star;
        const int64_t j0 = tile * BK_TILE;
        const float* frow = flux + star * N;
        for (int u = tid; u < BK_TILE + W - 1; u += BK_THREADS) {
            float x = 0.f;
            const bool ok = load_sample(nullptr, frow, N, j0 - h + u, x);
            xs[u] = ok ? x : qnan;
        }
        __syncthreads();
        for (int p = warp; p < BK_TILE && j0 + p < N; p += BK_WARPS) {
            const float med = median[star * N + j0 + p];
            float res = med;
            if (med == med) {
                /* the lane's samples, centred on the median (exact to fp32 for Eq. 4 as sum w x' / sum w); invalid -> NaN for now */
                float x[KPL];
#pragma unroll
                for (int i = 0; i < KPL; ++i) {
                    const int o = lane + 32 * i;
                    x[i] = (o < W) ? xs[p + o] - med : qnan;
                }
                /* Phase 2 (Eq. 1) */
                float ss = 0.f, cnt = 0.f;
#pragma unroll
                for (int i = 0; i < KPL; ++i)
                    if (x[i] > 0.f) { ss = fmaf(x[i], x[i], ss); cnt += 1.f; }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    ss += __shfl_xor_sync(0xFFFFFFFFu, ss, o);
                    cnt += __shfl_xor_sync(0xFFFFFFFFu, cnt, o);
                }
                float s = 0.f;
                bool on = cnt > 0.f;
                if (on) { s = SCALE_CONST * sqrtf(ss / cnt); on = s > 0.f; }
                if (on) {
                    const float cs = c * s, k = 1.f / cs;
                    /* invalid samples: far enough below for weight exactly 0 in every pass (mu stays within c s of the data) */
                    const float far = -1.0e3f * cs;
#pragma unroll
                    for (int i = 0; i < KPL; ++i) x[i] = (x[i] == x[i]) ? x[i] : far;
                    float mu = 0.f;                                 /* offset from the median */
                    const f32x2 na2 = pack2(nalpha, nalpha), kn2 = pack2(-k, -k);
                    for (int it = 0; it < n_iter; ++it) {
                        const float c0 = mu * k;                    /* -u = x(-k) + mu k */
                        const f32x2 cn2 = pack2(c0, c0);
                        f32x2 S2 = pack2(0.f, 0.f), R2 = S2;
#pragma unroll
                        for (int i = 0; i < KPL; i += 2) eval_weight_pair<APOW>(pack2(x[i], x[i + 1]), kn2, cn2, na2, S2, R2);
                        float S0, S1, R0, R1;
                        unpack2(S2, S0, S1);
                        unpack2(R2, R0, R1);
                        float Sw = S0 + S1, Rw = -(R0 + R1);        /* the pairs summed w*(-u) */
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) {
                            Sw += __shfl_xor_sync(0xFFFFFFFFu, Sw, o);
                            Rw += __shfl_xor_sync(0xFFFFFFFFu, Rw, o);
                        }
                        if (Sw > 0.f) mu = fmaf(Rw / Sw, cs, mu);   /* Eq. 4 */
                    }
                    res = med + mu;
                }
            }
            if (lane == 0) out[star * N + j0 + p] = res;
        }
        __syncthreads();
    }
}

/* ------------------------------------------------------------------ (0) the paper's design: a thread per position */
template <int WMAX>
__global__ void __launch_bounds__(128)
bk_paper_design(const float* __restrict__ flux, int64_t N, int64_t total, int W, int min_valid, float alpha, float c, int n_iter,
                float* __restrict__ out)
{
    const int h = (W - 1) >> 1;
    const float qnan = __int_as_float(0x7FC00000);
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t star = idx / N, p = idx - star * N;
        const float* frow = flux + star * N;
        float win[WMAX];                                            /* the thread's private copy of its window */
        int n = 0;
        for (int64_t j = p - h; j <= p + h; ++j) {
            float x = 0.f;
            if (load_sample(nullptr, frow, N, j, x)) win[n++] = x;
        }
        float own = 0.f;
        const bool own_ok = load_sample(nullptr, frow, N, p, own);
        if (!own_ok || n < min_valid || n == 0) { out[idx] = qnan; continue; }
        /* quickselect (Hoare partition) for rank k = (n-1)/2 */
        const int k = (n - 1) >> 1;
        int lo = 0, hi = n - 1;
        while (lo < hi) {
            const float pivot = win[(lo + hi) >> 1];
            int i = lo, j = hi;
            while (i <= j) {
                while (win[i] < pivot) ++i;
                while (win[j] > pivot) --j;
                if (i <= j) { const float t = win[i]; win[i] = win[j]; win[j] = t; ++i; --j; }
            }
            if (k <= j) hi = j; else if (k >= i) lo = i; else break;
        }
        const float med = win[k] + 0.f;
        float ss = 0.f, cnt = 0.f;
        for (int i = 0; i < n; ++i) {
            const float d = win[i] - med;
            if (d > 0.f) { ss = fmaf(d, d, ss); cnt += 1.f; }
        }
        float mu = med;
        if (cnt > 0.f) {
            const float s = SCALE_CONST * sqrtf(ss / cnt);
            if (s > 0.f) {
                const float cs = c * s, kk = 1.f / cs;
                for (int it = 0; it < n_iter; ++it) {
                    float S = 0.f, R = 0.f;
                    for (int i = 0; i < n; ++i) {
                        const float u = (win[i] - mu) * kk;
                        const float e = u < 0.f ? -alpha * u : u;
                        const float t = fmaxf(1.f - e * e, 0.f);
                        const float w = t * t;
                        S += w;
                        R = fmaf(w, u, R);
                    }
                    if (S > 0.f) mu = fmaf(R / S, cs, mu);
                }
            }
        }
        out[idx] = mu;
    }
}

int kpl_for(int W) { return (W + 31) / 32; }

} // namespace

extern "C" {

/* All pointers DEVICE; [n_stars, n_cadences] fp32 row-major; enqueue on `stream`, no synchronisation.
   Return 0, 1 (bad argument / window not compiled: W odd, 51 <= W <= 2176), or 3 (CUDA error). */
int umi_bakeoff_median_radix(const float* flux, int64_t n_stars, int64_t n_cadences, int W, float* median_out, void* stream)
{
    if (!flux || !median_out || n_stars < 0 || n_cadences < 0 || W < 51 || !(W & 1) || W > 2176) return 1;
    if (n_stars == 0 || n_cadences == 0) return 0;
    const int64_t tps = (n_cadences + BK_TILE - 1) / BK_TILE, nb = n_stars * tps;
    const unsigned grid = (unsigned)(nb < BK_MAX_GRID ? nb : BK_MAX_GRID);
    const size_t smem = (size_t)((BK_TILE + W - 1 + 3) & ~3) * 4 + (size_t)BK_WARPS * 256 * 4;
    const int mv = W / 3 > 1 ? W / 3 : 1;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int kpl = kpl_for(W);
    if (kpl <= 7) bk_median_radix<7><<<grid, BK_THREADS, smem, s>>>(flux, n_cadences, tps, nb, W, mv, median_out);
    else if (kpl <= 12) bk_median_radix<12><<<grid, BK_THREADS, smem, s>>>(flux, n_cadences, tps, nb, W, mv, median_out);
    else if (kpl <= 34) bk_median_radix<34><<<grid, BK_THREADS, smem, s>>>(flux, n_cadences, tps, nb, W, mv, median_out);
    else bk_median_radix<68><<<grid, BK_THREADS, smem, s>>>(flux, n_cadences, tps, nb, W, mv, median_out);
    return cudaGetLastError() == cudaSuccess ? 0 : 3;
}

int umi_bakeoff_median_warp_sorted(const float* flux, int64_t n_stars, int64_t n_cadences, int W, int run, float* median_out, void* stream)
{
    if (!flux || !median_out || n_stars < 0 || n_cadences < 0 || W < 51 || !(W & 1) || W > 2176 || run < 1) return 1;
    if (n_stars == 0 || n_cadences == 0) return 0;
    const int64_t rps = (n_cadences + run - 1) / run, nr = n_stars * rps;
    const int64_t ctas = (nr + 3) / 4;
    const unsigned grid = (unsigned)(ctas < BK_MAX_GRID ? ctas : BK_MAX_GRID);
    const int mv = W / 3 > 1 ? W / 3 : 1;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int kpl = kpl_for(W);
    if (kpl <= 7) bk_median_warp_sorted<7><<<grid, 128, 0, s>>>(flux, n_cadences, rps, nr, run, W, mv, median_out);
    else if (kpl <= 12) bk_median_warp_sorted<12><<<grid, 128, 0, s>>>(flux, n_cadences, rps, nr, run, W, mv, median_out);
    else if (kpl <= 34) bk_median_warp_sorted<34><<<grid, 128, 0, s>>>(flux, n_cadences, rps, nr, run, W, mv, median_out);
    else bk_median_warp_sorted<68><<<grid, 128, 0, s>>>(flux, n_cadences, rps, nr, run, W, mv, median_out);
    return cudaGetLastError() == cudaSuccess ? 0 : 3;
}

/* (0): W <= 385 (a private window of 385 floats per thread) */
int umi_bakeoff_paper_design(const float* flux, int64_t n_stars, int64_t n_cadences, int W, float alpha, float c, int n_iter,
                             float* trend_out, void* stream)
{
    if (!flux || !trend_out || n_stars < 0 || n_cadences < 0 || W < 1 || !(W & 1) || W > 385 || n_iter < 0) return 1;
    if (n_stars == 0 || n_cadences == 0) return 0;
    const int64_t total = n_stars * n_cadences;
    int64_t ctas = (total + 127) / 128;
    if (ctas > 148 * 64) ctas = 148 * 64;
    const int mv = W / 3 > 1 ? W / 3 : 1;
    bk_paper_design<385><<<(unsigned)ctas, 128, 0, static_cast<cudaStream_t>(stream)>>>(flux, n_cadences, total, W, mv, alpha, c, n_iter,
                                                                                   trend_out);
    return cudaGetLastError() == cudaSuccess ? 0 : 3;
}

/* median: the Phase-1 result (umi_detrend with n_iter = 0): NaN where the position has no trend */
int umi_bakeoff_reweight_warp_window(const float* flux, const float* median, int64_t n_stars, int64_t n_cadences, int W,
                                     float alpha, float c, int n_iter, float* trend_out, void* stream)
{
    if (!flux || !median || !trend_out || n_stars < 0 || n_cadences < 0 || W < 51 || !(W & 1) || W > 2176 || n_iter < 0) return 1;
    if (n_stars == 0 || n_cadences == 0) return 0;
    const int64_t tps = (n_cadences + BK_TILE - 1) / BK_TILE, nb = n_stars * tps;
    const unsigned grid = (unsigned)(nb < BK_MAX_GRID ? nb : BK_MAX_GRID);
    const size_t smem = (size_t)(BK_TILE + W - 1) * 4;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int kpl = kpl_for(W);
    const bool a2 = alpha == 2.f;
#define BK_LAUNCH(KPL)                                                                                                   \
    do {                                                                                                                 \
        if (a2) bk_reweight_warp_window<KPL, 1><<<grid, BK_THREADS, smem, s>>>(flux, median, n_cadences, tps, nb, W, alpha, c, n_iter, trend_out); \
        else bk_reweight_warp_window<KPL, -1><<<grid, BK_THREADS, smem, s>>>(flux, median, n_cadences, tps, nb, W, alpha, c, n_iter, trend_out);   \
    } while (0)
    if (kpl <= 8) BK_LAUNCH(8);
    else if (kpl <= 12) BK_LAUNCH(12);
    else if (kpl <= 34) BK_LAUNCH(34);
    else BK_LAUNCH(68);
#undef BK_LAUNCH
    return cudaGetLastError() == cudaSuccess ? 0 : 3;
}

} /* extern "C" */
