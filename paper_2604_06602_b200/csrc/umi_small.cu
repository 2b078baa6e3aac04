/*
 * umi_small.cu -- all three phases in one kernel for short windows
 * (W <= 49; Kepler / K2 / TESS-FFI 30-minute cadence gives W = 25).
 *
 * For a short window the per-tile sort of umi_median.cu costs more than the window itself, so
 * everything here runs in registers (a compile-time WT >= W wires, fully unrolled).
 *
 * Every WARP owns tiles of its own: 128 consecutive positions of one star (a thread owns 4
 * consecutive positions and the WT + 3 samples their windows share), staged with their halo into
 * the warp's private slice of shared memory -- no CTA-wide barrier anywhere.
 *
 * W == WT (the compiled lengths 9, 17, 25, 33, 49): ONE path for every warp, gaps and row ends
 * included.  Invalid slots (non-finite flux or time, outside the row: R2, R3, R16) are staged as
 * -inf / +inf ALTERNATELY along the tile.  A window then holds k invalid slots of which floor(k/2)
 * or ceil(k/2) are -inf, so the median of its n = WT - k valid samples -- rank (n-1)/2, the lower
 * middle (R6) -- sits at rank M = (WT-1)/2 of the padded window, or at rank M - 1 when k is odd and
 * the window got one -inf too few; both ranks come out of the same network:
 *   Phase 1  the WT - 3 samples the 4 windows share are sorted ONCE (Batcher odd-even merge
 *            network; only ranks m-4 .. m of it are read, m = (WT-1)/2, so most of it is dead
 *            code); rank M of window q is the 4th smallest of core ranks m-3 .. m and the window's
 *            own 3 samples e0 <= e1 <= e2:  min(C[m], max(C[m-1], e0), max(C[m-2], e1), max(C[m-3], e2)),
 *            rank M - 1 the 3rd smallest of C[m-4 .. m-1] and the same three.
 *   Phase 2/3 the arithmetic of umi_reweight.cu on the registers, invalid samples replaced by the
 *            per-tile sentinel (never above a median, weight exactly 0); the passes run on
 *            register-aligned sample pairs with packed FFMA2 / FMUL2 / FADD2.
 * W < WT (any other odd length): one position at a time through a full WT-wire network with the
 * missing wires padded (small_position); it re-reads its window from shared memory in every phase
 * instead of holding a second copy in registers, so no build of this file uses local memory.
 * Nothing here is shared with oracle/.
 */
#include <type_traits>
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

/* three values ascending */
__device__ __forceinline__ void sort3(float& a, float& b, float& c)
{
    float t = fminf(a, b); b = fmaxf(a, b); a = t;
    t = fminf(b, c); c = fmaxf(b, c); b = t;
    t = fminf(a, b); b = fmaxf(a, b); a = t;
}

/* one scalar (sample, position) evaluation of Eq. 2-4: accumulates sum w and sum w*u */
template <bool WELSCH>
__device__ __forceinline__ void eval_u(float x, float k, float c0k, float nalpha, float& S, float& R)
{
    const float u = fmaf(x, k, c0k);
    const float e = fmaxf(u, u * nalpha);                           /* |u_eff| */
    float w;
    if constexpr (WELSCH) {
        w = exp2f(e * e * -1.4426950408889634f);                    /* (R22) exp(-u_eff^2) */
    } else {
        const float t = __saturatef(fmaf(-e, e, 1.f));
        w = t * t;
    }
    S += w;
    R = fmaf(w, u, R);
}

/*
 * One position, any W <= WT (the path of window lengths that are not a compiled WT): the window is
 * win[0 .. W) in shared memory, invalid slots hold +-inf.  The W samples and WT - W missing wires go
 * through a full WT-wire network, the WT - n wires without a valid sample padded -inf for the first
 * (WT - n + 1)/2 of them and +inf for the rest, which puts rank (n-1)/2 of the valid samples (R6) in
 * the middle.  Later phases read the window again from shared memory.  FAMILY: sibling estimators (F4).
 */
template <int WT, bool FAMILY>
__device__ __noinline__ void small_position(const float* win, int W, float sent, const ReweightParams& prm,
                                            int min_valid, bool in_row, int64_t gidx)
{
    const int h = (W - 1) >> 1;
    const float nalpha = -prm.alpha;
    const float qnan = __int_as_float(0x7FC00000);
    auto sample = [&](int i, bool& ok) {                            /* wire i: value and validity */
        const float x = (i < W) ? win[i] : INFINITY;
        ok = finite_f32(x);
        return x;
    };

    /* ---- Phase 1 ---- */
    float a[WT];
    int n = 0;
#pragma unroll
    for (int i = 0; i < WT; ++i) {
        bool ok;
        (void)sample(i, ok);
        n += ok ? 1 : 0;
    }
    {
        const int n_low = (WT - n + 1) >> 1;                        /* wires sent to -inf */
        int seen = 0;
#pragma unroll
        for (int i = 0; i < WT; ++i) {
            bool ok;
            const float x = sample(i, ok);
            a[i] = ok ? x : ((seen < n_low) ? -INFINITY : INFINITY);
            seen += ok ? 0 : 1;
        }
    }
    batcher_sort<WT>(a);
    float med = a[(WT - 1) / 2];
    med += 0.f;                                                     /* -0.0 -> +0.0 (R18) */
    bool own_ok;
    (void)sample(h, own_ok);
    const bool has = in_row && own_ok && n >= min_valid && n > 0;   /* (R4, R5) */

    /* mu is carried as an unevaluated pair hi + lo, and every residual is formed as (x - mu_hi) - mu_lo: the subtraction is
       exact for the samples near mu, which are the ones that carry weight, wherever mu ends up -- next to the median (then
       one ulp of a single fp32 mu, 6e-8 of the flux, would be ~2e-5 in units of u, which an expanding iteration amplifies:
       heavy ties under alpha = 10, c = 2.5 with 9 passes gave 1.8e-5 in one of 3,000 random cases) or far from it (two valid
       samples {-9999, 4.0}, min_valid = 1: the median is -9999 and the passes converge on 4.0006).  One more subtraction per
       evaluation: this is the path that can afford it. */
    float mu = med, mu_lo = 0.f;
    const bool want_scale = FAMILY && prm.scale_out != nullptr;
    if ((prm.n_iter > 0 || want_scale) && has) {
        bool on;
        float s = 0.f;
        if (FAMILY && prm.scale_kind == SCALE_MAD) {
            /* ---- MAD (R21): rank (n-1)/2 of the n absolute deviations, same padding ---- */
            const int n_low = (WT - n + 1) >> 1;
            int seen = 0;
#pragma unroll
            for (int i = 0; i < WT; ++i) {
                bool ok;
                const float x = sample(i, ok);
                a[i] = ok ? fabsf(x - med) : ((seen < n_low) ? -INFINITY : INFINITY);
                seen += ok ? 0 : 1;
            }
            batcher_sort<WT>(a);
            s = a[(WT - 1) / 2];
            on = s > 0.f;
        } else {
            /* ---- Phase 2 (Eq. 1) ---- */
            float ss = 0.f, cnt = 0.f;
            for (int i = 0; i < W; ++i) {
                const float x = win[i];
                const float d = (finite_f32(x) ? x : sent) - med;
                if (d > 0.f) {
                    ss = fmaf(d, d, ss);
                    cnt += 1.f;
                }
            }
            on = cnt > 0.f;                                         /* (R8) */
            if (on) {
                s = SCALE_CONST * sqrtf(ss / cnt);
                on = s > 0.f;
            }
        }
        if (want_scale) prm.scale_out[gidx] = s;
        const float cs = on ? prm.c * s : 0.f;
        const float k = on ? 1.f / cs : 0.f;
        /* ---- Phase 3 (Eq. 2-4) ---- */
        for (int it = 0; it < prm.n_iter; ++it) {
            const float c0 = -mu_lo * k;
            float S = 0.f, R = 0.f;
            for (int i = 0; i < W; ++i) {
                const float xr = win[i];
                const float x = (finite_f32(xr) ? xr : sent) - mu;
                if (FAMILY && prm.weight_kind == WEIGHT_WELSCH) eval_u<true>(x, k, c0, nalpha, S, R);
                else eval_u<false>(x, k, c0, nalpha, S, R);
            }
            if (on && S > 0.f) {                                    /* Eq. 4; (R11): (mu, mu_lo) += cs R / S, error-free */
                const float step = (R / S) * cs;
                const float t = mu + step, bb = t - mu;
                const float lo = ((mu - (t - bb)) + (step - bb)) + mu_lo;
                mu = t + lo;
                mu_lo = lo - (mu - t);
            }
        }
    } else if (want_scale && in_row) {
        prm.scale_out[gidx] = qnan;
    }
    if (in_row) {
        const float tr = mu;                                        /* hi of the normalised pair = fl(hi + lo) */
        prm.out[gidx] = has ? tr : qnan;
        if (prm.flat != nullptr)                                    /* PAPER.md:155 normalisation */
            prm.flat[gidx] = has ? win[h] / tr : qnan;
    }
}

} // namespace

/* resident CTAs per SM the register allocation aims at: 6 for W = 25 (80 registers, nothing spilled; measured 5.30 ms on
   2,000 config-3 stars against 5.38 with the compiler's own choice of 96 registers and 5.34 at 7 CTAs; the alpha = 2
   build: 4 / 5 / 6 / 7 / 8 CTAs = 5.16 / 5.02 / 4.89 / 4.98 / 5.02 ms); the longer windows
   hold WT + 3 samples per thread and get the registers they need */
constexpr int ks_min_ctas(int wt, bool family) { return wt <= 9 ? 6 : wt <= 17 ? 5 : wt <= 25 ? (family ? 5 : 6) : wt <= 33 ? 4 : 3; }

template <int WT, bool FAMILY, int APOW>
__global__ void __launch_bounds__(KS_THREADS, ks_min_ctas(WT, FAMILY))
umi_small_kernel(const __grid_constant__ ReweightParams prm, int min_valid)   /* (__grid_constant__: small_position takes prm by reference) */
{
    constexpr int NSAMP = WT + 3;                                   /* multiple of 4 (WT = 1 mod 8) */
    constexpr int M = (WT - 1) / 2;                                 /* half window = middle rank; a multiple of 4 */
    constexpr int NXS = KS_WARP_TILE + NSAMP;                       /* staged floats per warp */
    using mask_t = typename std::conditional<(NSAMP <= 32), uint32_t, uint64_t>::type;
    constexpr mask_t WMASK = (mask_t)((((uint64_t)1) << WT) - 1);

    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    float* xs = reinterpret_cast<float*>(smem_raw) + warp * NXS;    /* this warp's slice */
    const int W = prm.W;                                            /* odd, <= WT */
    const int h = (W - 1) >> 1;
    const float nalpha = -prm.alpha;
    const float qnan = __int_as_float(0x7FC00000);
    const bool vec = (prm.N & 3) == 0 && (reinterpret_cast<uintptr_t>(prm.flux) & 15) == 0 &&
                     (reinterpret_cast<uintptr_t>(prm.time) & 15) == 0;

    for (int64_t bid = (int64_t)blockIdx.x * KS_WARPS + warp; bid < prm.n_blocks; bid += (int64_t)gridDim.x * KS_WARPS) {
        const int64_t star = bid / prm.tiles_per_star;
        const int64_t tile = bid - star * prm.tiles_per_star;
        const int64_t j0 = tile * KS_WARP_TILE;
        const int64_t jbase = j0 - M;                               /* cadence of staged index 0 (a multiple of 4) */
        const float* frow = prm.flux + star * prm.N;
        const double* trow = prm.time ? prm.time + star * prm.N : nullptr;

        /* stage; invalid slots become -inf, +inf, -inf, ... in staged order; tile min / max of the valid samples */
        float tmin = INFINITY, tmax = -INFINITY;
        int n_inv = 0;                                              /* invalid slots so far (the same in every lane) */
        if (vec) {
            for (int u0 = 0; u0 < NXS; u0 += 128) {
                const int u = u0 + 4 * lane;
                const int64_t j = jbase + u;
                float4 v = make_float4(qnan, qnan, qnan, qnan);
                if (u < NXS && j >= 0 && j < prm.N) {               /* a group of 4 lies entirely inside or outside the row */
                    v = __ldg(reinterpret_cast<const float4*>(frow + j));
                    if (trow != nullptr) {
                        const double2 ta = __ldg(reinterpret_cast<const double2*>(trow + j));
                        const double2 tb = __ldg(reinterpret_cast<const double2*>(trow + j + 2));
                        if (!finite_f64(ta.x)) v.x = qnan;
                        if (!finite_f64(ta.y)) v.y = qnan;
                        if (!finite_f64(tb.x)) v.z = qnan;
                        if (!finite_f64(tb.y)) v.w = qnan;
                    }
                }
                const bool live = u < NXS;                          /* (the last round is partial) */
                const bool b0 = live && !finite_f32(v.x), b1 = live && !finite_f32(v.y), b2 = live && !finite_f32(v.z), b3 = live && !finite_f32(v.w);
                const int mine = (int)b0 + (int)b1 + (int)b2 + (int)b3;
                int incl = mine;                                    /* inclusive scan over the lanes */
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int t = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                    if (lane >= o) incl += t;
                }
                int ord = n_inv + incl - mine;                      /* ordinal of this lane's first invalid slot */
                n_inv += __shfl_sync(0xFFFFFFFFu, incl, 31);
                if (b0) { v.x = (ord & 1) ? INFINITY : -INFINITY; ++ord; } else { tmin = fminf(tmin, v.x); tmax = fmaxf(tmax, v.x); }   /* (fminf / fmaxf skip the NaN of a dead lane) */
                if (b1) { v.y = (ord & 1) ? INFINITY : -INFINITY; ++ord; } else { tmin = fminf(tmin, v.y); tmax = fmaxf(tmax, v.y); }
                if (b2) { v.z = (ord & 1) ? INFINITY : -INFINITY; ++ord; } else { tmin = fminf(tmin, v.z); tmax = fmaxf(tmax, v.z); }
                if (b3) { v.w = (ord & 1) ? INFINITY : -INFINITY; ++ord; } else { tmin = fminf(tmin, v.w); tmax = fmaxf(tmax, v.w); }
                if (u < NXS) *reinterpret_cast<float4*>(xs + u) = v;
            }
        } else {
            for (int u0 = 0; u0 < NXS; u0 += 32) {
                const int u = u0 + lane;
                float x = 0.f;
                const bool ok = u < NXS && load_sample(trow, frow, prm.N, jbase + u, x);
                const unsigned bad = __ballot_sync(0xFFFFFFFFu, u < NXS && !ok);
                const int ord = n_inv + __popc(bad & ((1u << lane) - 1u));
                n_inv += __popc(bad);
                if (ok) { tmin = fminf(tmin, x); tmax = fmaxf(tmax, x); }
                else x = (ord & 1) ? INFINITY : -INFINITY;
                if (u < NXS) xs[u] = x;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            tmin = fminf(tmin, __shfl_xor_sync(0xFFFFFFFFu, tmin, o));
            tmax = fmaxf(tmax, __shfl_xor_sync(0xFFFFFFFFu, tmax, o));
        }
        __syncwarp();
        float sent = 0.f;                                           /* DESIGN.md, "Sentinel" */
        if (tmin <= tmax) {
            if constexpr (!FAMILY)
                sent = tmin - (2.f * SCALE_CONST) * prm.c_over_alpha * (tmax - tmin);
            else   /* s <= tmax - tmin for either scale; Welsch needs |u_eff| >= 16 for an exact 0 */
                sent = tmin - (prm.weight_kind == WEIGHT_WELSCH ? 24.f : 2.f) * prm.c_over_alpha * (tmax - tmin);
            sent = fmaxf(sent, -3.0e38f);
        }
        const bool clean = (n_inv == 0);                            /* every staged slot valid (and inside the row) */
        const int64_t jq = j0 + 4 * lane;                           /* first of the thread's 4 positions */

        if (W != WT) {
            /* a window length without a compiled network of its own: one position at a time; position jl's
               window [jl - h, jl + h] sits at staged [jl + M - h, jl + M + h] */
#pragma unroll 1
            for (int q = 0; q < 4; ++q)
                small_position<WT, FAMILY>(xs + 4 * lane + q + (M - h), W, sent, prm, min_valid, jq + q < prm.N,
                                           star * prm.N + jq + q);
            __syncwarp();
            continue;
        }

        float s[NSAMP];
#pragma unroll
        for (int g = 0; g < NSAMP / 4; ++g) {
            const float4 v = reinterpret_cast<const float4*>(xs)[lane + g];
            s[4 * g] = v.x; s[4 * g + 1] = v.y; s[4 * g + 2] = v.z; s[4 * g + 3] = v.w;
        }
        /* ---- Phase 1: shared core s[3 .. WT), sorted once; its ranks M-4 .. M ---- */
        float c4, c3, c2, c1, c0;                                   /* core ranks M, M-1, M-2, M-3, M-4 */
        {
            float core[WT - 3];
#pragma unroll
            for (int i = 0; i < WT - 3; ++i) core[i] = s[3 + i];
            batcher_sort<WT - 3>(core);
            c4 = core[M]; c3 = core[M - 1]; c2 = core[M - 2]; c1 = core[M - 3]; c0 = core[M - 4];
        }
        mask_t inv = 0;                                             /* bit i: s[i] is an invalid slot */
        mask_t neg = 0;                                             /* bit i: ... staged as -inf */
        if (!clean) {
#pragma unroll
            for (int i = 0; i < NSAMP; ++i) {
                inv |= finite_f32(s[i]) ? (mask_t)0 : ((mask_t)1 << i);
                neg |= (s[i] == -INFINITY) ? ((mask_t)1 << i) : (mask_t)0;
            }
        }
        float med[4], mu[4];
        bool has[4];
        int nval[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            /* the 3 samples of window q outside the core: s[q .. 3) and s[WT .. WT + q) */
            float e0 = (q < 1) ? s[0] : s[WT + q - 1];
            float e1 = (q < 2) ? s[1] : s[WT + q - 2];
            float e2 = (q < 3) ? s[2] : s[WT + q - 3];
            sort3(e0, e1, e2);
            /* rank M of the padded window: 4th smallest of core ranks M-3 .. M and e0..e2 */
            float m = fminf(fminf(c4, fmaxf(c3, e0)), fminf(fmaxf(c2, e1), fmaxf(c1, e2)));
            nval[q] = WT;
            has[q] = WT >= min_valid;
            if (!clean) {
                int k, a;
                if constexpr (sizeof(mask_t) == 4) {
                    k = __popc((uint32_t)((inv >> q) & WMASK));
                    a = __popc((uint32_t)((neg >> q) & WMASK));
                } else {
                    k = __popcll((uint64_t)((inv >> q) & WMASK));
                    a = __popcll((uint64_t)((neg >> q) & WMASK));
                }
                /* k odd and one -inf short of ceil(k/2): the lower middle is one rank down, the 3rd smallest
                   of core ranks M-4 .. M-1 and e0..e2 */
                if ((k & 1) && 2 * a < k)
                    m = fminf(fminf(c3, fmaxf(c2, e0)), fminf(fmaxf(c1, e1), fmaxf(c0, e2)));
                nval[q] = WT - k;
                const bool own_ok = ((inv >> (q + M)) & 1) == 0;
                has[q] = own_ok && nval[q] >= min_valid && nval[q] > 0;        /* (R4, R5); outside the row = invalid own slot */
            }
            m += 0.f;                                               /* -0.0 -> +0.0 (R18) */
            med[q] = has[q] ? m : 0.f;
            mu[q] = med[q];
        }
        const float own[4] = {s[M], s[M + 1], s[M + 2], s[M + 3]};   /* the positions' own samples (for flux / trend) */
        /* From here on everything is CENTRED on one of the thread's own medians, the one of smallest magnitude (a robust
           reference, chosen as in umi_reweight.cu): x' = x - ref is exact for every sample that can carry weight, and mu
           is carried as an offset, so its fp32 rounding is relative to the residuals and not to the flux.  (On raw samples
           one ulp of mu is 6e-8 of the flux -- ~2e-5 in units of u -- which an expanding iteration, e.g. heavy ties under
           alpha = 10, c = 2.5 with 9 passes, amplifies; small_position has the case that was measured.) */
        float ref = 0.f, rabs = INFINITY;
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (has[q] && fabsf(med[q]) < rabs) { rabs = fabsf(med[q]); ref = med[q]; }
        const float xsent = sent - ref;
        if (!clean) {
#pragma unroll
            for (int i = 0; i < NSAMP; ++i) s[i] = ((inv >> i) & 1) ? xsent : s[i] - ref;
        } else {
            const f32x2 nref2 = pack2(-ref, -ref);                  /* NSAMP is even: register-aligned pairs, as the passes use them */
#pragma unroll
            for (int i = 0; i < NSAMP; i += 2) unpack2(fadd2(pack2(s[i], s[i + 1]), nref2), s[i], s[i + 1]);
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            med[q] = has[q] ? med[q] - ref : 0.f;
            mu[q] = med[q];
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
                    /* rank (n-1)/2 of the n deviations: the WT - n invalid wires padded -inf, then +inf */
                    float a[WT];
                    const int n_low = (WT - nval[q] + 1) >> 1;
                    int seen = 0;
#pragma unroll
                    for (int i = 0; i < WT; ++i) {
                        const bool bad = (inv >> (q + i)) & 1;
                        a[i] = bad ? ((seen < n_low) ? -INFINITY : INFINITY) : fabsf(s[q + i] - med[q]);
                        seen += bad ? 1 : 0;
                    }
                    batcher_sort<WT>(a);
                    sc = a[M];
                    on[q] = has[q] && sc > 0.f;
                } else {
                    float ss = 0.f, cnt = 0.f;
#pragma unroll
                    for (int i = 0; i < WT; ++i) {
                        const float d = s[q + i] - med[q];
                        if (d > 0.f) {                              /* one compare, two predicated updates */
                            ss = fmaf(d, d, ss);
                            cnt += 1.f;
                        }
                    }
                    on[q] = has[q] && cnt > 0.f;                    /* (R8) */
                    if (on[q]) {
                        sc = SCALE_CONST * sqrtf(ss / cnt);
                        on[q] = sc > 0.f;
                    }
                }
                if (want_scale && jq + q < prm.N) prm.scale_out[star * prm.N + jq + q] = has[q] ? sc : qnan;
                cs[q] = on[q] ? prm.c * sc : 0.f;
                k[q] = on[q] ? 1.f / cs[q] : 0.f;
            }
            /* APOW >= 0 (alpha = 2^APOW): the pairs form alpha*u by an integer add (umi_device.cuh), which would wrap an
               overflowed -u = k (mu - x) to a small value; warps in which it could overflow (|x|, |mu| <= amax; never seen
               on real data) take a rolled scalar loop over the staged window instead, which multiplies */
            bool risky = false;
            if constexpr (APOW >= 0) {
                const float amax = 4.f * fmaxf(fabsf(sent), fmaxf(fabsf(tmin), fabsf(tmax)));   /* |x - ref|, |mu - ref| <= 2 max|x| */
#pragma unroll
                for (int q = 0; q < 4; ++q) risky = risky || !(k[q] * amax < 1.2676506e30f);   /* 2^100 */
                risky = __any_sync(0xFFFFFFFFu, risky);
            }
            /* ---- Phase 3 (Eq. 2-4) ---- */
            for (int it = 0; it < prm.n_iter; ++it) {
                float S[4], R[4], c0k[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) { S[q] = 0.f; R[q] = 0.f; c0k[q] = -mu[q] * k[q]; }
                if (APOW >= 0 && risky) {
#pragma unroll 1
                    for (int i = 0; i < WT + 3; ++i) {
                        const float xr = xs[4 * lane + i];
                        const float x = finite_f32(xr) ? xr - ref : xsent;
#pragma unroll
                        for (int q = 0; q < 4; ++q)
                            if (i >= q && i < q + WT) eval_u<false>(x, k[q], c0k[q], nalpha, S[q], R[q]);
                    }
                } else if (FAMILY && prm.weight_kind == WEIGHT_WELSCH) {
#pragma unroll
                    for (int q = 0; q < 4; ++q)
#pragma unroll
                        for (int i = 0; i < WT; ++i) eval_u<true>(s[q + i], k[q], c0k[q], nalpha, S[q], R[q]);
                } else {
                    const f32x2 na2 = pack2(nalpha, nalpha);
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        /* the WT samples of window q as (WT-1)/2 register-aligned pairs + one single:
                           pairs start at an even index of s[], so q odd leaves s[q] over, q even s[q+WT-1] */
                        constexpr int NPAIR = (WT - 1) / 2;
                        const int first = q + (q & 1);
                        const f32x2 k2 = pack2(-k[q], -k[q]), c02 = pack2(-c0k[q], -c0k[q]);   /* pairs work on -u */
                        f32x2 Sa = pack2(0.f, 0.f), Ra = Sa;              /* one accumulator pair per position: the 4 positions interleave */
#pragma unroll
                        for (int j = 0; j < NPAIR; ++j)
                            eval_weight_pair<APOW>(pack2(s[first + 2 * j], s[first + 2 * j + 1]), k2, c02, na2, Sa, Ra);
                        float S0, S1, R0, R1;
                        unpack2(Sa, S0, S1);
                        unpack2(Ra, R0, R1);
                        S[q] = S0 + S1;
                        R[q] = -(R0 + R1);                          /* the pairs summed w*(-u) */
                    }
                    /* the samples left over, two positions to a packed evaluation (halves: position q, q + 1) */
#pragma unroll
                    for (int q = 0; q < 4; q += 2) {
                        const f32x2 x2 = pack2(s[q + WT - 1], s[q + 1]);
                        const f32x2 k2 = pack2(-k[q], -k[q + 1]), c02 = pack2(-c0k[q], -c0k[q + 1]);
                        f32x2 Sp = pack2(0.f, 0.f), Rp = Sp;
                        eval_weight_pair<APOW>(x2, k2, c02, na2, Sp, Rp);
                        float S0, S1, R0, R1;
                        unpack2(Sp, S0, S1);
                        unpack2(Rp, R0, R1);
                        S[q] += S0; S[q + 1] += S1;
                        R[q] -= R0; R[q + 1] -= R1;
                    }
                }
#pragma unroll
                for (int q = 0; q < 4; ++q)   /* Eq. 4; (R11).  R/S by reciprocal + multiply (2 ulp; S is in [w_min, WT]): the quotient only scales
                                                 the step cs*R/S, itself < 1e-2 of the flux, so the trend moves by < 1e-9 relative; an IEEE
                                                 division here is 10 of the ~190 instructions of a pass */
                    if (on[q] && S[q] > 0.f) mu[q] = fmaf(__fdividef(R[q], S[q]), cs[q], mu[q]);
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (jq + q < prm.N) {
                const int64_t gi = star * prm.N + jq + q;
                const float tr = mu[q] + ref;
                prm.out[gi] = has[q] ? tr : qnan;
                if (prm.flat != nullptr) prm.flat[gi] = has[q] ? own[q] / tr : qnan;   /* PAPER.md:155 normalisation */
            }
        }
        __syncwarp();                                               /* the slice is free for the next tile */
    }
}

template <bool FAMILY, int APOW>
static cudaError_t launch_small_t(const ReweightParams& prm, int min_valid, int wt, unsigned grid, cudaStream_t stream)
{
    const size_t smem = (size_t)KS_WARPS * (size_t)(KS_WARP_TILE + wt + 3) * sizeof(float);
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
    /* the paper's default alpha = 2 takes the build that forms alpha*u by an integer add on the bit pattern (umi_device.cuh):
       5 instead of 6 FMA-pipe lane-operations per evaluation, 5.12 -> 4.86 ms on 2,000 config-3 stars.  (Round 1 measured no
       gain from it on the CTA-tile kernel with its second unrolled copy of the passes; here the guard is a rolled loop.) */
    if (family) return launch_small_t<true, -1>(prm, min_valid, wt, grid, stream);
    if (alpha_pow2(prm.alpha) == 1) return launch_small_t<false, 1>(prm, min_valid, wt, grid, stream);
    return launch_small_t<false, -1>(prm, min_valid, wt, grid, stream);
}

} // namespace umi
