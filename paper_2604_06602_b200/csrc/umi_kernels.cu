/*
 * umi_kernels.cu -- sm_100a kernels of the UMI sliding-window detrender.
 *
 * Method: arxiv/paper_2604_06602, section 2 (lines 33-63); readings
 * R1..R18 in DESIGN.md.  Nothing here is shared with oracle/.
 *
 * Two kernels per umi_detrend call ("Kernels"):
 *
 *  umi_median_kernel (Phase 1)
 *    CTA = one star x one tile of T consecutive positions.  The T windows of a
 *    tile live inside one union of U = T + W - 1 samples.  The union is sorted
 *    ONCE per tile (bitonic, shared memory, 64-bit key|index), then each lane
 *    of one warp walks T/32 consecutive positions, keeping the union-rank of
 *    the current window's median: a slide removes one sample and adds one, so
 *    the median moves by at most a couple of included ranks.  Exact (the
 *    result is a selected sample), O(log^2 U) per position for the sort plus
 *    O(1) expected per slide, instead of O(W) per position for a per-thread
 *    quickselect.
 *
 *  umi_reweight_kernel (Phase 2 + Phase 3, Eq. 1-4)
 *    CTA = one star x 512 positions; a thread owns 4 consecutive positions and
 *    streams the W+3 samples they share from shared memory with one 128-bit
 *    load per 16 (sample, position) evaluations; all accumulators stay in
 *    registers, no reductions.  Invalid samples are replaced in shared memory
 *    by a finite per-tile sentinel far below the tile minimum, which Eq. 1
 *    never counts and Eq. 3 always gives weight 0, so the inner loop carries no
 *    validity predicate.
 */
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "umi_internal.h"

namespace umi {

namespace {

constexpr uint32_t KEY_INVALID = 0xFFFFFFFFu;
constexpr float SCALE_CONST = 0.6745f;

/* Order-preserving float -> uint32 key; -0.0 is folded onto +0.0 (R18). */
__device__ __forceinline__ uint32_t float_to_key(float x)
{
    uint32_t b = __float_as_uint(x);
    if (b == 0x80000000u) b = 0u;
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

__device__ __forceinline__ float key_to_float(uint32_t k)
{
    uint32_t b = (k & 0x80000000u) ? (k & 0x7FFFFFFFu) : ~k;
    return __uint_as_float(b);
}

__device__ __forceinline__ bool finite_f32(float x)
{
    return (__float_as_uint(x) & 0x7F800000u) != 0x7F800000u;
}

__device__ __forceinline__ bool finite_f64(double t)
{
    return ((uint32_t)__double2hiint(t) & 0x7FF00000u) != 0x7FF00000u;
}

/* (R2, R3, R16) one slot of one star row: in range, finite flux, finite time. */
__device__ __forceinline__ bool load_sample(const double* __restrict__ trow,
                                            const float* __restrict__ frow,
                                            int64_t N, int64_t j, float& x)
{
    if (j < 0 || j >= N) return false;
    x = __ldg(frow + j);
    bool ok = finite_f32(x);
    if (trow != nullptr) ok = ok && finite_f64(__ldg(trow + j));
    return ok;
}

} // namespace

/* ===================================================================== Phase 1 */

__global__ void __launch_bounds__(K1_THREADS)
umi_median_kernel(MedianParams prm)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int NS = prm.NS;
    const int W = prm.W;
    const int T = prm.T;
    const int h = (W - 1) >> 1;
    uint64_t* srt = reinterpret_cast<uint64_t*>(smem_raw);          /* [NS] key<<32 | union index */
    float* medbuf = reinterpret_cast<float*>(srt + NS);             /* [NS] (first T used) */
    uint16_t* rank = reinterpret_cast<uint16_t*>(medbuf + NS);      /* [NS] union index -> rank */
    __shared__ int s_nvu;

    const int tid = threadIdx.x;

    for (int64_t bid = blockIdx.x; bid < prm.n_blocks; bid += gridDim.x) {
        const int64_t star = bid / prm.tiles_per_star;
        const int64_t tile = bid - star * prm.tiles_per_star;
        const int64_t j0 = tile * T;                                /* first position of the tile */
        const int64_t jbase = j0 - h;                               /* cadence of union index 0 */
        const int64_t rem = prm.N - j0;
        const int Tact = rem < T ? (int)rem : T;
        const float* frow = prm.flux + star * prm.N;
        const double* trow = prm.time ? prm.time + star * prm.N : nullptr;

        if (tid == 0) s_nvu = 0;

        /* stage: union index u <-> cadence jbase + u; U = T + W - 1 == NS */
        for (int u = tid; u < NS; u += K1_THREADS) {
            float x = 0.f;
            bool ok = load_sample(trow, frow, prm.N, jbase + u, x);
            uint32_t key = ok ? float_to_key(x) : KEY_INVALID;
            srt[u] = ((uint64_t)key << 32) | (uint32_t)u;
        }
        __syncthreads();

        /* bitonic sort, ascending; keys are unique because the index is part of them */
        for (int k = 2; k <= NS; k <<= 1) {
            for (int j = k >> 1; j > 0; j >>= 1) {
                for (int t = tid; t < (NS >> 1); t += K1_THREADS) {
                    const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                    const int p = i | j;
                    const bool up = ((i & k) == 0);
                    const uint64_t a = srt[i], b = srt[p];
                    if ((a > b) == up) { srt[i] = b; srt[p] = a; }
                }
                __syncthreads();
            }
        }

        /* ranks and the number of valid samples in the union */
        for (int r = tid; r < NS; r += K1_THREADS) {
            const uint64_t e = srt[r];
            rank[(uint32_t)e] = (uint16_t)r;
            const bool v = (uint32_t)(e >> 32) != KEY_INVALID;
            const bool vnext = (r + 1 < NS) && ((uint32_t)(srt[r + 1] >> 32) != KEY_INVALID);
            if (v && !vnext) s_nvu = r + 1;
        }
        __syncthreads();
        const int nvu = s_nvu;

        /* walk: one warp, lane w owns positions [w*Ts, (w+1)*Ts) of the tile */
        if (tid < 32) {
            const int Ts = (Tact + 31) >> 5;
            int pbeg = tid * Ts;
            int pend = pbeg + Ts;
            if (pend > Tact) pend = Tact;
            const bool lane_on = pbeg < pend;
            if (!lane_on) pbeg = 0;
            const uint32_t uW = (uint32_t)W;

            /* n = valid samples in window pbeg = union [pbeg, pbeg + W) */
            int n = 0;
            for (int t = 0; t < W; ++t) n += (rank[pbeg + t] < nvu) ? 1 : 0;
            const int k0 = (n - 1) >> 1;                            /* (R6) lower median */
            int rho = -1;
            {
                int acc = 0;
                for (int r = 0; r < nvu; ++r) {
                    const uint32_t u = (uint32_t)srt[r];
                    const bool inc = (u - (uint32_t)pbeg) < uW;
                    acc += inc ? 1 : 0;
                    if (inc && acc == k0 + 1) rho = r;
                }
            }
            if (lane_on) {
                int p = pbeg;
                for (;;) {
                    /* emit position p (R4, R5) */
                    const bool own = rank[p + h] < nvu;
                    float m = __int_as_float(0x7FC00000);
                    if (own && n >= prm.min_valid && n > 0)
                        m = key_to_float((uint32_t)(srt[rho] >> 32));
                    medbuf[p] = m;
                    if (++p >= pend) break;
                    /* slide to window p: union index p-1 leaves, p+W-1 enters */
                    const int ro = rank[p - 1], ri = rank[p + W - 1];
                    const bool vo = ro < nvu, vi = ri < nvu;
                    const int n2 = n - (vo ? 1 : 0) + (vi ? 1 : 0);
                    if (n2 == 0) {
                        rho = -1;
                    } else if (n == 0) {
                        rho = ri;
                    } else {
                        const int k2 = (n2 - 1) >> 1;
                        int below = ((n - 1) >> 1) - ((vo && ro < rho) ? 1 : 0) + ((vi && ri < rho) ? 1 : 0);
                        const uint32_t up = (uint32_t)p;
                        if (vo && ro == rho) {
                            int r = rho + 1;
                            while (r < nvu && ((uint32_t)srt[r] - up) >= uW) ++r;
                            if (r < nvu) {
                                rho = r;
                            } else {
                                r = rho - 1;
                                while (r > 0 && ((uint32_t)srt[r] - up) >= uW) --r;
                                rho = r;
                                --below;
                            }
                        }
                        while (below > k2) {
                            int r = rho - 1;
                            while (r > 0 && ((uint32_t)srt[r] - up) >= uW) --r;
                            rho = r;
                            --below;
                        }
                        while (below < k2) {
                            int r = rho + 1;
                            while (r < nvu - 1 && ((uint32_t)srt[r] - up) >= uW) ++r;
                            rho = r;
                            ++below;
                        }
                    }
                    n = n2;
                }
            }
        }
        __syncthreads();

        float* orow = prm.out + star * prm.N + j0;
        for (int p = tid; p < Tact; p += K1_THREADS) orow[p] = medbuf[p];
        __syncthreads();
    }
}

/* ============================================================= Phase 2 + Phase 3 */

namespace {

struct PosState {
    float med, mu, k, c0, cs, S, R;
    bool active;
};

/* Phase 2, Eq. 1: strictly-above-median residuals (R7). */
__device__ __forceinline__ void eval_scale(float x, float med, float& ss, float& cnt)
{
    const float d = x - med;
    const float dp = fmaxf(d, 0.f);
    ss = fmaf(dp, dp, ss);
    cnt += (d > 0.f) ? 1.f : 0.f;
}

/* Phase 3, Eq. 2-3 on u = (x - mu)/(c s) = x*k + c0; accumulates sum w and sum w*u. */
__device__ __forceinline__ void eval_weight(float x, float k, float c0, float nalpha,
                                            float& S, float& R)
{
    const float a = fmaf(x, k, c0);          /* u */
    const float b = a * nalpha;              /* -alpha*u */
    const float e = fmaxf(a, b);             /* |u_eff| for either sign, any alpha > 0 */
    float t = fmaf(-e, e, 1.f);
    t = fmaxf(t, 0.f);                       /* (R12) */
    const float w = t * t;
    S += w;
    R = fmaf(w, a, R);
}

} // namespace

__global__ void __launch_bounds__(K2_THREADS)
umi_reweight_kernel(ReweightParams prm)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* xs = reinterpret_cast<float*>(smem_raw);
    __shared__ float s_red[2 * (K2_THREADS / 32)];

    const int tid = threadIdx.x;
    const int W = prm.W;
    const int h = (W - 1) >> 1;
    const int hal = (h + 3) & ~3;
    const int delta = hal - h;
    const int G = (3 + delta + 2 * h) / 4 + 1;          /* float4 groups per thread */
    const int nx = K2_TILE + 4 * G;                     /* staged floats */
    const int g_lo = (3 + delta + 3) >> 2;              /* first group fully inside all 4 windows */
    const int g_hi = (delta + 2 * h - 3) >= 0 ? ((delta + 2 * h - 3) >> 2) : -1;   /* last such group */
    const float nalpha = -prm.alpha;
    const float qnan = __int_as_float(0x7FC00000);

    for (int64_t bid = blockIdx.x; bid < prm.n_blocks; bid += gridDim.x) {
        const int64_t star = bid / prm.tiles_per_star;
        const int64_t tile = bid - star * prm.tiles_per_star;
        const int64_t j0 = tile * K2_TILE;
        const int64_t jbase = j0 - hal;
        const float* frow = prm.flux + star * prm.N;
        const double* trow = prm.time ? prm.time + star * prm.N : nullptr;
        float* orow = prm.out + star * prm.N;

        /* stage the union, NaN marks invalid; tile min / max of the valid samples */
        float tmin = INFINITY, tmax = -INFINITY;
        for (int u = tid; u < nx; u += K2_THREADS) {
            float x = 0.f;
            const bool ok = load_sample(trow, frow, prm.N, jbase + u, x);
            if (ok) { tmin = fminf(tmin, x); tmax = fmaxf(tmax, x); }
            xs[u] = ok ? x : qnan;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            tmin = fminf(tmin, __shfl_xor_sync(0xFFFFFFFFu, tmin, o));
            tmax = fmaxf(tmax, __shfl_xor_sync(0xFFFFFFFFu, tmax, o));
        }
        if ((tid & 31) == 0) { s_red[(tid >> 5) * 2] = tmin; s_red[(tid >> 5) * 2 + 1] = tmax; }
        __syncthreads();
#pragma unroll
        for (int w = 0; w < K2_THREADS / 32; ++w) {
            tmin = fminf(tmin, s_red[2 * w]);
            tmax = fmaxf(tmax, s_red[2 * w + 1]);
        }
        /* sentinel: alpha*(mu - x)/(c s) >= 2 for every window of the tile, since
           mu >= tmin and s <= 0.6745 (tmax - tmin)  ("Sentinel") */
        float sent = 0.f;
        if (tmin <= tmax) {
            sent = tmin - 2.f * (prm.c * SCALE_CONST / prm.alpha) * (tmax - tmin);
            sent = fmaxf(sent, -3.0e38f);
        }
        for (int u = tid; u < nx; u += K2_THREADS) {
            const float x = xs[u];
            if (x != x) xs[u] = sent;
        }
        __syncthreads();

        /* per-position state: 4 consecutive positions, local index 4*tid + q */
        float med[K2_NPOS], mu[K2_NPOS], kk[K2_NPOS], cs[K2_NPOS];
        bool act[K2_NPOS];
        bool any_act = false;
#pragma unroll
        for (int q = 0; q < K2_NPOS; ++q) {
            const int64_t j = j0 + 4 * tid + q;
            med[q] = (j < prm.N) ? orow[j] : qnan;
            act[q] = (med[q] == med[q]);
            any_act = any_act || act[q];
            mu[q] = act[q] ? med[q] : 0.f;
            kk[q] = 0.f;
            cs[q] = 0.f;
        }
        const float4* xs4 = reinterpret_cast<const float4*>(xs) + tid;

        if (__any_sync(0xFFFFFFFFu, any_act)) {
            /* ---- Phase 2 ---- */
            float ss[K2_NPOS], cnt[K2_NPOS];
#pragma unroll
            for (int q = 0; q < K2_NPOS; ++q) { ss[q] = 0.f; cnt[q] = 0.f; }
            for (int g = 0; g < G; ++g) {
                const float4 v = xs4[g];
                const float xv[4] = {v.x, v.y, v.z, v.w};
                if (g >= g_lo && g <= g_hi) {
#pragma unroll
                    for (int q = 0; q < K2_NPOS; ++q)
#pragma unroll
                        for (int r = 0; r < 4; ++r) eval_scale(xv[r], mu[q], ss[q], cnt[q]);
                } else {
#pragma unroll
                    for (int q = 0; q < K2_NPOS; ++q)
#pragma unroll
                        for (int r = 0; r < 4; ++r) {
                            const int o = 4 * g + r - delta - q;
                            if (o >= 0 && o <= 2 * h) eval_scale(xv[r], mu[q], ss[q], cnt[q]);
                        }
                }
            }
#pragma unroll
            for (int q = 0; q < K2_NPOS; ++q) {
                bool on = act[q] && cnt[q] > 0.f;                   /* (R8) */
                float s = 0.f;
                if (on) {
                    s = SCALE_CONST * sqrtf(ss[q] / cnt[q]);
                    on = s > 0.f;
                }
                act[q] = on;
                cs[q] = on ? prm.c * s : 0.f;
                kk[q] = on ? 1.f / cs[q] : 0.f;
            }

            /* ---- Phase 3 ---- */
            for (int it = 0; it < prm.n_iter; ++it) {
                float S[K2_NPOS], R[K2_NPOS], c0[K2_NPOS];
#pragma unroll
                for (int q = 0; q < K2_NPOS; ++q) { S[q] = 0.f; R[q] = 0.f; c0[q] = -mu[q] * kk[q]; }
                for (int g = 0; g < G; ++g) {
                    const float4 v = xs4[g];
                    const float xv[4] = {v.x, v.y, v.z, v.w};
                    if (g >= g_lo && g <= g_hi) {
#pragma unroll
                        for (int q = 0; q < K2_NPOS; ++q)
#pragma unroll
                            for (int r = 0; r < 4; ++r) eval_weight(xv[r], kk[q], c0[q], nalpha, S[q], R[q]);
                    } else {
#pragma unroll
                        for (int q = 0; q < K2_NPOS; ++q)
#pragma unroll
                            for (int r = 0; r < 4; ++r) {
                                const int o = 4 * g + r - delta - q;
                                if (o >= 0 && o <= 2 * h) eval_weight(xv[r], kk[q], c0[q], nalpha, S[q], R[q]);
                            }
                    }
                }
#pragma unroll
                for (int q = 0; q < K2_NPOS; ++q)
                    if (act[q] && S[q] > 0.f) mu[q] = fmaf(R[q] / S[q], cs[q], mu[q]);   /* Eq. 4; (R11) */
            }
        }

#pragma unroll
        for (int q = 0; q < K2_NPOS; ++q) {
            const int64_t j = j0 + 4 * tid + q;
            if (j < prm.N && med[q] == med[q]) orow[j] = mu[q];
        }
        __syncthreads();
    }
}

} // namespace umi
