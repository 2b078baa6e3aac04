/*
 * umi_small.cu -- all three phases in one kernel for short windows
 * (W <= 49; Kepler / K2 / TESS-FFI 30-minute cadence gives W = 25).
 *
 * For a short window the per-tile sort of umi_median.cu costs more than the window
 * itself, so here one thread owns one position and keeps its whole window in
 * registers (a compile-time WT >= W wires, fully unrolled, no local memory):
 *   Phase 1  Batcher odd-even merge network on the WT wires; only the middle output is
 *            used, so the compiler drops every min/max that cannot reach it (202 of
 *            280 for WT = 25).  The network delivers the fixed rank (WT-1)/2; the
 *            median of the n valid samples has rank (n-1)/2 (R6), so the WT-n invalid
 *            or padding wires are set to -inf for the first (WT-n+1)/2 of them and to
 *            +inf for the rest, which moves the wanted rank to the middle.  Warps whose
 *            32 windows are all valid (the common case) skip that bookkeeping.
 *   Phase 2/3 the same arithmetic as umi_reweight.cu on the 25 registers, invalid
 *            wires replaced by the per-tile sentinel (weight exactly 0, never above the
 *            median).
 * CTA = 256 consecutive positions of one star; tile + halo staged in shared memory.
 * Nothing here is shared with oracle/.
 */
#include <utility>

#include "umi_device.cuh"

namespace umi {

namespace {

/* Batcher's odd-even merge sort for arbitrary N as a compile-time list of compare-exchanges. */
template <int N>
struct BatcherNet {
    int count;
    short lo[N * 12], hi[N * 12];
};

template <int N>
__host__ __device__ constexpr BatcherNet<N> make_batcher()
{
    BatcherNet<N> net{};
    int c = 0;
    for (int p = 1; p < N; p <<= 1)
        for (int k = p; k >= 1; k >>= 1)
            for (int j = k % p; j + k < N; j += 2 * k)
                for (int i = 0; i < k && i < N - j - k; ++i)
                    if ((i + j) / (2 * p) == (i + j + k) / (2 * p)) {
                        net.lo[c] = (short)(i + j);
                        net.hi[c] = (short)(i + j + k);
                        ++c;
                    }
    net.count = c;
    return net;
}

template <int N, int I>
__device__ __forceinline__ void batcher_step(float (&a)[N])
{
    constexpr BatcherNet<N> net = make_batcher<N>();
    if constexpr (I < net.count) {
        constexpr int i = net.lo[I], j = net.hi[I];
        const float lo = fminf(a[i], a[j]);
        const float hi = fmaxf(a[i], a[j]);
        a[i] = lo;
        a[j] = hi;
    }
}

template <int N, int... I>
__device__ __forceinline__ void batcher_apply(float (&a)[N], std::integer_sequence<int, I...>)
{
    (batcher_step<N, I>(a), ...);
}

/* Sorts a[] ascending; outputs that are never read cost nothing (dead-code elimination). */
template <int N>
__device__ __forceinline__ void batcher_sort(float (&a)[N])
{
    batcher_apply<N>(a, std::make_integer_sequence<int, N * 12>{});
}

} // namespace

/* FAMILY = false: the paper's path.  true: sibling estimators (F4): MAD scale by a second network
   on the absolute deviations (R21), Welsch weights (R22), optional scale output. */
template <int WT, bool FAMILY>
__global__ void __launch_bounds__(KS_THREADS)
umi_small_kernel(ReweightParams prm, int min_valid)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* xs = reinterpret_cast<float*>(smem_raw);                 /* [KS_THREADS + WT - 1] */
    __shared__ float s_red[2 * (KS_THREADS / 32)];

    const int tid = threadIdx.x;
    const int W = prm.W;                                            /* odd, <= WT */
    const int h = (W - 1) >> 1;
    const int nx = KS_THREADS + WT - 1;
    const float nalpha = -prm.alpha;
    const float qnan = __int_as_float(0x7FC00000);

    for (int64_t bid = blockIdx.x; bid < prm.n_blocks; bid += gridDim.x) {
        const int64_t star = bid / prm.tiles_per_star;
        const int64_t tile = bid - star * prm.tiles_per_star;
        const int64_t j0 = tile * KS_THREADS;
        const int64_t jbase = j0 - h;                               /* cadence of staged index 0 */
        const float* frow = prm.flux + star * prm.N;
        const double* trow = prm.time ? prm.time + star * prm.N : nullptr;
        float* orow = prm.out + star * prm.N;

        /* stage; NaN marks invalid; tile min / max of the valid samples */
        float tmin = INFINITY, tmax = -INFINITY;
        for (int u = tid; u < nx; u += KS_THREADS) {
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
        for (int w = 0; w < KS_THREADS / 32; ++w) {
            tmin = fminf(tmin, s_red[2 * w]);
            tmax = fmaxf(tmax, s_red[2 * w + 1]);
        }
        float sent = 0.f;                                           /* DESIGN.md, "Sentinel" */
        if (tmin <= tmax) {
            if constexpr (!FAMILY)
                sent = tmin - 2.f * (prm.c * SCALE_CONST / prm.alpha) * (tmax - tmin);
            else   /* s <= tmax - tmin for either scale; Welsch needs |u_eff| >= 16 for an exact 0 */
                sent = tmin - (prm.weight_kind == WEIGHT_WELSCH ? 24.f : 2.f) * (prm.c / prm.alpha) * (tmax - tmin);
            sent = fmaxf(sent, -3.0e38f);
        }

        /* window of position j0 + tid: staged indices tid .. tid + W - 1 */
        float x[WT];
        bool all_ok = (W == WT);
#pragma unroll
        for (int i = 0; i < WT; ++i) {
            x[i] = (i < W) ? xs[tid + i] : qnan;
            all_ok = all_ok && (x[i] == x[i]);
        }
        const int64_t j = j0 + tid;
        const bool in_row = j < prm.N;

        /* ---- Phase 1 ---- */
        float a[WT];
        int n = WT;
        bool own_ok = true;
        uint64_t okmask = ~0ull;                                    /* FAMILY: which wires are valid */
        if (__all_sync(0xFFFFFFFFu, all_ok)) {
#pragma unroll
            for (int i = 0; i < WT; ++i) a[i] = x[i];
        } else {
            n = 0;
#pragma unroll
            for (int i = 0; i < WT; ++i) n += (x[i] == x[i]) ? 1 : 0;
            const int n_low = (WT - n + 1) >> 1;                    /* wires sent to -inf */
            int seen = 0;
            own_ok = false;
#pragma unroll
            for (int i = 0; i < WT; ++i) {
                const bool ok = (x[i] == x[i]);
                if (i == h) own_ok = ok && (i < W);
                a[i] = ok ? x[i] : ((seen < n_low) ? -INFINITY : INFINITY);
                seen += ok ? 0 : 1;
                if (!ok) okmask &= ~(1ull << i);
                x[i] = ok ? x[i] : sent;
            }
        }
        batcher_sort<WT>(a);
        float med = a[(WT - 1) / 2];
        med += 0.f;                                                 /* -0.0 -> +0.0 (R18) */
        const bool has = in_row && own_ok && n >= min_valid && n > 0;   /* (R4, R5) */

        float mu = med;
        const bool want_scale = FAMILY && prm.scale_out != nullptr;
        if ((prm.n_iter > 0 || want_scale) && __any_sync(0xFFFFFFFFu, has)) {
            bool on;
            float s = 0.f;
            if (FAMILY && prm.scale_kind == SCALE_MAD) {
                /* ---- MAD (R21): rank (n-1)/2 of the n absolute deviations, same padding trick ---- */
                const int n_low = (WT - n + 1) >> 1;
                int seen = 0;
#pragma unroll
                for (int i = 0; i < WT; ++i) {
                    const bool ok = (okmask >> i) & 1ull;
                    a[i] = ok ? fabsf(x[i] - med) : ((seen < n_low) ? -INFINITY : INFINITY);
                    seen += ok ? 0 : 1;
                }
                batcher_sort<WT>(a);
                s = a[(WT - 1) / 2];
                on = has && s > 0.f;
            } else {
            /* ---- Phase 2 (Eq. 1) ---- */
            float ss = 0.f, cnt = 0.f;
#pragma unroll
            for (int i = 0; i < WT; ++i) {
                const float d = x[i] - med;
                const float dp = fmaxf(d, 0.f);
                ss = fmaf(dp, dp, ss);
                cnt += (d > 0.f) ? 1.f : 0.f;
            }
            on = has && cnt > 0.f;                                  /* (R8) */
            if (on) {
                s = SCALE_CONST * sqrtf(ss / cnt);
                on = s > 0.f;
            }
            }
            if (want_scale && in_row) prm.scale_out[star * prm.N + j] = has ? s : qnan;
            const float cs = on ? prm.c * s : 0.f;
            const float k = on ? 1.f / cs : 0.f;
            /* ---- Phase 3 (Eq. 2-4) ---- */
            for (int it = 0; it < prm.n_iter; ++it) {
                const float c0 = -mu * k;
                float S0 = 0.f, S1 = 0.f, R0 = 0.f, R1 = 0.f;
#pragma unroll
                for (int i = 0; i < WT; ++i) {
                    const float u = fmaf(x[i], k, c0);
                    const float b = u * nalpha;
                    const float e = fmaxf(u, b);
                    float w;
                    if (FAMILY && prm.weight_kind == WEIGHT_WELSCH) {
                        w = exp2f(e * e * -1.4426950408889634f);    /* (R22) exp(-u_eff^2) */
                    } else {
                        const float t = __saturatef(fmaf(-e, e, 1.f));
                        w = t * t;
                    }
                    if (i & 1) { S1 += w; R1 = fmaf(w, u, R1); }
                    else       { S0 += w; R0 = fmaf(w, u, R0); }
                }
                const float S = S0 + S1, R = R0 + R1;
                if (on && S > 0.f) mu = fmaf(R / S, cs, mu);        /* Eq. 4; (R11) */
            }
        }
        if (want_scale && in_row && !has) prm.scale_out[star * prm.N + j] = qnan;
        if (in_row) {
            orow[j] = has ? mu : qnan;
            if (prm.flat != nullptr)                                /* PAPER.md:155 normalisation */
                prm.flat[star * prm.N + j] = has ? xs[tid + h] / mu : qnan;
        }
        __syncthreads();
    }
}

template <bool FAMILY>
static cudaError_t launch_small_t(const ReweightParams& prm, int min_valid, int wt, unsigned grid, cudaStream_t stream)
{
    const size_t smem = (size_t)(KS_THREADS + wt - 1) * sizeof(float);
    switch (wt) {
    case 9: umi_small_kernel<9, FAMILY><<<grid, KS_THREADS, smem, stream>>>(prm, min_valid); break;
    case 17: umi_small_kernel<17, FAMILY><<<grid, KS_THREADS, smem, stream>>>(prm, min_valid); break;
    case 25: umi_small_kernel<25, FAMILY><<<grid, KS_THREADS, smem, stream>>>(prm, min_valid); break;
    case 33: umi_small_kernel<33, FAMILY><<<grid, KS_THREADS, smem, stream>>>(prm, min_valid); break;
    case 49: umi_small_kernel<49, FAMILY><<<grid, KS_THREADS, smem, stream>>>(prm, min_valid); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_small(const ReweightParams& prm, bool family, int min_valid, int wt, unsigned grid, cudaStream_t stream)
{
    return family ? launch_small_t<true>(prm, min_valid, wt, grid, stream)
                  : launch_small_t<false>(prm, min_valid, wt, grid, stream);
}

} // namespace umi
