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

/*
 * One position, general case (any number of valid samples, W <= WT): the window is read from
 * shared memory at win[0 .. W).  FAMILY = false: the paper's path.  true: sibling estimators
 * (F4): MAD scale by a second network on the absolute deviations (R21), Welsch weights (R22),
 * optional scale output.  Called by all 32 lanes together (it votes).
 */
template <int WT, bool FAMILY>
__device__ __noinline__ void small_position(const float* win, int W, float sent, const ReweightParams& prm,
                                            int min_valid, bool in_row, int64_t gidx)
{
    const int h = (W - 1) >> 1;
    const float nalpha = -prm.alpha;
    const float qnan = __int_as_float(0x7FC00000);
    float x[WT];
    bool all_ok = (W == WT);
#pragma unroll
    for (int i = 0; i < WT; ++i) {
        x[i] = (i < W) ? win[i] : qnan;
        all_ok = all_ok && (x[i] == x[i]);
    }

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
        if (want_scale && in_row) prm.scale_out[gidx] = has ? s : qnan;
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
    if (want_scale && in_row && !has) prm.scale_out[gidx] = qnan;
    if (in_row) {
        prm.out[gidx] = has ? mu : qnan;
        if (prm.flat != nullptr)                                /* PAPER.md:155 normalisation */
            prm.flat[gidx] = has ? win[h] / mu : qnan;
    }
}

/* three values ascending */
__device__ __forceinline__ void sort3(float& a, float& b, float& c)
{
    float t = fminf(a, b); b = fmaxf(a, b); a = t;
    t = fminf(b, c); c = fmaxf(b, c); b = t;
    t = fminf(a, b); b = fmaxf(a, b); a = t;
}

/*
 * CTA = KS_TILE = 4 * KS_THREADS consecutive positions of one star; a thread owns 4 consecutive
 * positions and the WT + 3 samples their windows share.
 *
 * Fast path (the paper's estimator, W == WT, every one of the thread's WT + 3 samples valid, decided
 * per warp): the 4 windows have WT - 3 samples in common.  That core is sorted ONCE (only its
 * ranks m-3 .. m are kept, m = (WT-1)/2, so most of the network is dead code); the median of a
 * window is the 4th smallest of those four core values and its own 3 remaining samples:
 *     med = min(C[m], max(C[m-1], e0), max(C[m-2], e1), max(C[m-3], e2)),   e0 <= e1 <= e2
 * (the m-3 core values below C[m-3] are below everything that can be the answer).  Phases 2-3 then
 * run on the registers, 4 independent positions interleaved.
 * Any other case goes through small_position, one position at a time.
 */
template <int WT, bool FAMILY, int APOW>
__global__ void __launch_bounds__(KS_THREADS)
umi_small_kernel(ReweightParams prm, int min_valid)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* xs = reinterpret_cast<float*>(smem_raw);                 /* [KS_TILE + WT - 1] */
    __shared__ float s_red[2 * (KS_THREADS / 32)];

    constexpr int NSAMP = WT + 3;                                   /* multiple of 4 (WT = 1 mod 8) */
    constexpr int M = (WT - 1) / 2;
    const int tid = threadIdx.x;
    const int W = prm.W;                                            /* odd, <= WT */
    const int h = (W - 1) >> 1;
    const int nx = KS_TILE + WT - 1;
    const float nalpha = -prm.alpha;
    const float qnan = __int_as_float(0x7FC00000);

    for (int64_t bid = blockIdx.x; bid < prm.n_blocks; bid += gridDim.x) {
        const int64_t star = bid / prm.tiles_per_star;
        const int64_t tile = bid - star * prm.tiles_per_star;
        const int64_t j0 = tile * KS_TILE;
        const int64_t jbase = j0 - h;                               /* cadence of staged index 0 */
        const float* frow = prm.flux + star * prm.N;
        const double* trow = prm.time ? prm.time + star * prm.N : nullptr;

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
                sent = tmin - (2.f * SCALE_CONST) * prm.c_over_alpha * (tmax - tmin);
            else   /* s <= tmax - tmin for either scale; Welsch needs |u_eff| >= 16 for an exact 0 */
                sent = tmin - (prm.weight_kind == WEIGHT_WELSCH ? 24.f : 2.f) * prm.c_over_alpha * (tmax - tmin);
            sent = fmaxf(sent, -3.0e38f);
        }

        const int64_t jq = j0 + 4 * tid;                            /* first of the thread's 4 positions */
        bool fast = false;
        {
            if (W == WT) {
                /* all WT + 3 samples valid <=> all 4 windows complete (and inside the row) */
                bool ok = true;
#pragma unroll
                for (int g = 0; g < NSAMP / 4; ++g) {
                    const float4 v = reinterpret_cast<const float4*>(xs)[tid + g];
                    ok = ok && (v.x == v.x) && (v.y == v.y) && (v.z == v.z) && (v.w == v.w);
                }
                fast = __all_sync(0xFFFFFFFFu, ok) && WT >= min_valid;
            }
        }
        if (fast) {
            float s[NSAMP];
#pragma unroll
            for (int g = 0; g < NSAMP / 4; ++g) {
                const float4 v = reinterpret_cast<const float4*>(xs)[tid + g];
                s[4 * g] = v.x; s[4 * g + 1] = v.y; s[4 * g + 2] = v.z; s[4 * g + 3] = v.w;
            }
            /* ---- Phase 1: shared core s[3 .. WT), sorted once ---- */
            float core[WT - 3];
#pragma unroll
            for (int i = 0; i < WT - 3; ++i) core[i] = s[3 + i];
            batcher_sort<WT - 3>(core);
            const float c0 = core[M - 3], c1 = core[M - 2], c2 = core[M - 1], c3 = core[M];
            float med[4], mu[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                /* the 3 samples of window q outside the core: s[q .. 3) and s[WT .. WT + q) */
                float e0 = (q < 1) ? s[0] : s[WT + q - 1];
                float e1 = (q < 2) ? s[1] : s[WT + q - 2];
                float e2 = (q < 3) ? s[2] : s[WT + q - 3];
                sort3(e0, e1, e2);
                float m = fminf(fminf(c3, fmaxf(c2, e0)), fminf(fmaxf(c1, e1), fmaxf(c0, e2)));
                m += 0.f;                                           /* -0.0 -> +0.0 (R18) */
                med[q] = m;
                mu[q] = m;
            }
            const bool want_scale = FAMILY && prm.scale_out != nullptr;
            if (prm.n_iter > 0 || want_scale) {
                /* ---- Phase 2 (Eq. 1), or the MAD (R21) for the sibling estimators ---- */
                float cs[4], k[4];
                bool on[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    float sc = 0.f;
                    if (FAMILY && prm.scale_kind == SCALE_MAD) {
                        float a[WT];
#pragma unroll
                        for (int i = 0; i < WT; ++i) a[i] = fabsf(s[q + i] - med[q]);
                        batcher_sort<WT>(a);
                        sc = a[M];
                        on[q] = sc > 0.f;
                    } else {
                        float ss = 0.f, cnt = 0.f;
#pragma unroll
                        for (int i = 0; i < WT; ++i) {
                            const float d = s[q + i] - med[q];
                            if (d > 0.f) {                          /* one compare, two predicated updates */
                                ss = fmaf(d, d, ss);
                                cnt += 1.f;
                            }
                        }
                        on[q] = cnt > 0.f;                          /* (R8) */
                        if (on[q]) {
                            sc = SCALE_CONST * sqrtf(ss / cnt);
                            on[q] = sc > 0.f;
                        }
                    }
                    if (want_scale) prm.scale_out[star * prm.N + jq + q] = sc;
                    cs[q] = on[q] ? prm.c * sc : 0.f;
                    k[q] = on[q] ? 1.f / cs[q] : 0.f;
                }
                /* APOW >= 0 (alpha = 2^APOW): the pairs form alpha*u by an integer add (umi_device.cuh) unless
                   -u = k (mu - x) could overflow somewhere in the warp; |x|, |mu| <= max(|tmin|, |tmax|) */
                bool risky = false;
                if constexpr (APOW >= 0) {
                    const float amax = fmaxf(fabsf(tmin), fabsf(tmax));
#pragma unroll
                    for (int q = 0; q < 4; ++q) risky = risky || !(k[q] * amax < 1.2676506e30f);   /* 2^100 */
                    risky = __any_sync(0xFFFFFFFFu, risky);
                }
                /* ---- Phase 3 (Eq. 2-4) ---- */
                for (int it = 0; it < prm.n_iter; ++it) {
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const float c0k = -mu[q] * k[q];
                        if (FAMILY && prm.weight_kind == WEIGHT_WELSCH) {
                            float S = 0.f, R = 0.f;
#pragma unroll
                            for (int i = 0; i < WT; ++i) {
                                const float u = fmaf(s[q + i], k[q], c0k);
                                const float e = fmaxf(u, u * nalpha);
                                const float w = exp2f(e * e * -1.4426950408889634f);   /* (R22) exp(-u_eff^2) */
                                S += w;
                                R = fmaf(w, u, R);
                            }
                            if (on[q] && S > 0.f) mu[q] = fmaf(R / S, cs[q], mu[q]);
                            continue;
                        }
                        /* the WT samples of window q as (WT-1)/2 register-aligned pairs + one single:
                           pairs start at an even index of s[], so q odd peels s[q], q even peels s[q+WT-1] */
                        constexpr int NPAIR = (WT - 1) / 2;
                        const int first = q + (q & 1);
                        const f32x2 k2 = pack2(-k[q], -k[q]), c02 = pack2(-c0k, -c0k), na2 = pack2(nalpha, nalpha);   /* pairs work on -u */
                        f32x2 Sa = pack2(0.f, 0.f), Sb = Sa, Ra = Sa, Rb = Sa;
                        if (APOW >= 0 && !risky) {
#pragma unroll
                            for (int j = 0; j < NPAIR; ++j) {
                                const f32x2 x2 = pack2(s[first + 2 * j], s[first + 2 * j + 1]);
                                if (j & 1) eval_weight_pair<APOW>(x2, k2, c02, na2, Sb, Rb);
                                else       eval_weight_pair<APOW>(x2, k2, c02, na2, Sa, Ra);
                            }
                        } else {
#pragma unroll
                            for (int j = 0; j < NPAIR; ++j) {
                                const f32x2 x2 = pack2(s[first + 2 * j], s[first + 2 * j + 1]);
                                if (j & 1) eval_weight_pair<-1>(x2, k2, c02, na2, Sb, Rb);
                                else       eval_weight_pair<-1>(x2, k2, c02, na2, Sa, Ra);
                            }
                        }
                        float S0, S1, R0, R1;
                        unpack2(fadd2(Sa, Sb), S0, S1);
                        unpack2(fadd2(Ra, Rb), R0, R1);
                        R0 = -R0;                                   /* the pairs summed w*(-u) */
                        R1 = -R1;
                        {
                            const float xs1 = (q & 1) ? s[q] : s[q + WT - 1];
                            const float u = fmaf(xs1, k[q], c0k);
                            const float e = fmaxf(u, u * nalpha);
                            const float t = __saturatef(fmaf(-e, e, 1.f));
                            const float w = t * t;
                            S0 += w;
                            R0 = fmaf(w, u, R0);
                        }
                        const float S = S0 + S1, R = R0 + R1;
                        if (on[q] && S > 0.f) mu[q] = fmaf(R / S, cs[q], mu[q]);   /* Eq. 4; (R11) */
                    }
                }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int64_t gi = star * prm.N + jq + q;
                prm.out[gi] = mu[q];
                if (prm.flat != nullptr) prm.flat[gi] = s[q + M] / mu[q];   /* PAPER.md:155 normalisation */
            }
        } else {
#pragma unroll 1
            for (int q = 0; q < 4; ++q)
                small_position<WT, FAMILY>(xs + 4 * tid + q, W, sent, prm, min_valid, jq + q < prm.N,
                                           star * prm.N + jq + q);
        }
        __syncthreads();
    }
}

template <bool FAMILY, int APOW>
static cudaError_t launch_small_t(const ReweightParams& prm, int min_valid, int wt, unsigned grid, cudaStream_t stream)
{
    const size_t smem = (size_t)(KS_TILE + wt - 1) * sizeof(float);
    switch (wt) {
    case 9: umi_small_kernel<9, FAMILY, APOW><<<grid, KS_THREADS, smem, stream>>>(prm, min_valid); break;
    case 17: umi_small_kernel<17, FAMILY, APOW><<<grid, KS_THREADS, smem, stream>>>(prm, min_valid); break;
    case 25: umi_small_kernel<25, FAMILY, APOW><<<grid, KS_THREADS, smem, stream>>>(prm, min_valid); break;
    case 33: umi_small_kernel<33, FAMILY, APOW><<<grid, KS_THREADS, smem, stream>>>(prm, min_valid); break;
    case 49: umi_small_kernel<49, FAMILY, APOW><<<grid, KS_THREADS, smem, stream>>>(prm, min_valid); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_small(const ReweightParams& prm, bool family, int min_valid, int wt, unsigned grid, cudaStream_t stream)
{
    /* APOW stays -1 here: the integer-add form of alpha*u (umi_device.cuh) was measured on this kernel and is
       slower (config 3: 30.7 ms against 27.2 ms) -- its ALU pipe already carries the median network, and the
       second copy of the unrolled passes costs registers; the reweighting kernel is where it pays */
    return family ? launch_small_t<true, -1>(prm, min_valid, wt, grid, stream)
                  : launch_small_t<false, -1>(prm, min_valid, wt, grid, stream);
}

} // namespace umi
