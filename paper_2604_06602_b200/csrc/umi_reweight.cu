/*
 * umi_reweight.cu -- Phase 2 + Phase 3 (Eq. 1-4): upper-RMS scale and
 * n_iter asymmetric Tukey-bisquare passes, starting from the Phase-1 median.
 *
 * Every WARP owns tiles of its own: 128 consecutive positions of one star, a thread owning 4
 * consecutive positions.  The warp stages its tile and the W-1 halo into its private slice of
 * shared memory, so the kernel has no CTA-wide barrier at all (__syncwarp only) and a warp whose
 * tile lies in a gap does not hold the other three up.  A thread streams the W+3 samples its 4
 * windows share with one 128-bit load per 16 (sample, position) evaluations; all accumulators stay
 * in registers, there are no reductions.  Invalid samples are replaced in shared memory by a finite
 * per-tile sentinel far below the tile minimum, which Eq. 1 never counts and Eq. 3 always gives
 * weight 0, so the inner loop carries no validity predicate.
 *
 * What the median kernel hands over (umi_internal.h): one word per position = where in its window
 * the median sample sits | n+ << 16.  The median is read from the staged samples, n+ (Eq. 1's
 * count, exact on the sorted keys) leaves Phase 2 with a sum of squares only, and the staged
 * samples are centred on the mid-range of the tile's MEDIANS -- a robust reference: one wild
 * sample (a -9999 fill value, a 1e6 glitch) moves neither it nor the precision of the others.
 *
 * Inner loop: per (sample, position), on u' = -u
 *     u' = x*(-k) + mu*k            k = 1/(c s)
 *     -e = min(u', alpha*u, -1.0f)  as signed integers: -min(|u_eff|, 1), Eq. 2's case split and
 *                                   Eq. 3's cut-off (R12) in one DPX instruction; for alpha = 2^m
 *                                   alpha*u is an integer add on the bits of u' (no multiply)
 *     n  = e*e - 1  (<= 0);  w = n*n;  S += w;  R += w*x'            Eq. 4: mu' <- R/S
 * The fma/mul/add steps run as sm_100a packed fp32x2 instructions (FFMA2/FMUL2/FADD2) on two
 * consecutive samples at a time; the edge groups use the scalar float form of the same arithmetic.
 * Nothing here is shared with oracle/.
 */
#include "umi_device.cuh"

#ifndef UMI_K2_MIN_CTAS
#define UMI_K2_MIN_CTAS 5
#endif
#ifndef UMI_K2_MIN_CTAS_POW2
#define UMI_K2_MIN_CTAS_POW2 6     /* alpha = 2^m builds: 78 registers, no spills.  Measured (W = 361 / 2161 / 217, ms): 5 CTAs 7.20 / 48.7 / 8.16, 6 CTAs 7.21 / 49.2 / 8.07, 8 CTAs (64 registers, 8 bytes spilled per thread) 7.18 / 49.0 / 8.02 */
#endif
#ifndef UMI_K2_UNROLL
#define UMI_K2_UNROLL 8
#endif

namespace umi {

namespace {

constexpr int K2_UNROLL = UMI_K2_UNROLL;

/* Phase 2, Eq. 1: strictly-above-median residuals (R7). */
__device__ __forceinline__ void eval_scale(float x, float med, float& ss, float& cnt)
{
    const float d = x - med;
    if (d > 0.f) {                                   /* one compare, two predicated updates */
        ss = fmaf(d, d, ss);
        cnt += 1.f;
    }
}

/* Phase 3, one (sample, position): accumulates sum w and sum w*u. */
__device__ __forceinline__ void eval_weight(float x, float k, float c0, float nalpha,
                                            float& S, float& R)
{
    const float a = fmaf(x, k, c0);                  /* u */
    const float b = a * nalpha;                      /* -alpha*u */
    const float e = fmaxf(a, b);                     /* |u_eff| */
    const float t = __saturatef(fmaf(-e, e, 1.f));   /* FFMA.SAT */
    const float w = t * t;
    S += w;
    R = fmaf(w, x, R);                               /* sum w x (centred samples): Eq. 4's numerator */
}

/* Sibling weight (F4; R22): Welsch, w = exp(-u_eff^2), no cut-off. */
__device__ __forceinline__ void eval_welsch(float x, float k, float c0, float nalpha,
                                            float& S, float& R)
{
    const float a = fmaf(x, k, c0);                  /* u */
    const float e = fmaxf(a, a * nalpha);            /* |u_eff| */
    const float w = exp2f(e * e * -1.4426950408889634f);   /* exp(-e^2); 0 for the sentinel (e >= 16) */
    S += w;
    R = fmaf(w, x, R);
}

/* Phase 3 on one 128-bit group: 4 samples (two fp32x2 pairs) x 4 positions = 8 pair
   evaluations, written stage by stage so that the 8 dependency chains interleave.  x01[q], x23[q]: the group's
   two sample pairs as position q sees them (all four the same in an interior group; in an edge group the
   samples outside window q are replaced by the sentinel, whose weight is exactly 0).
   kn2 = (-k, -k), cn2 = (mu k, mu k): the group works on u' = -u.  Exactly one of u' and
   alpha*u = -alpha*u' is <= 0, and it is -|u_eff| of Eq. 2; as signed integers a non-positive float
   sorts below every positive one, and among non-positive floats the larger magnitude is the larger
   integer, so ONE three-input integer minimum (DPX VIMNMX3) with the bit pattern of -1.0f gives
   -min(|u_eff|, 1): Eq. 2's case split and Eq. 3's cut-off in a single ALU-pipe instruction
   (was: FMNMX for |u_eff| and a second FMNMX for the clamp).  1 - min(|u_eff|,1)^2 is then >= 0
   by construction, and bitwise the value max(1 - u_eff^2, 0) had. */
template <int APOW>
__device__ __forceinline__ void eval_weight_group(const f32x2 (&x01)[K2_NPOS], const f32x2 (&x23)[K2_NPOS],
                                                  const f32x2 (&kn2)[K2_NPOS], const f32x2 (&cn2)[K2_NPOS], f32x2 nalpha2,
                                                  f32x2 (&S2)[K2_NPOS], f32x2 (&R2)[K2_NPOS])
{
    f32x2 a2[2 * K2_NPOS], w2[2 * K2_NPOS];
#pragma unroll
    for (int q = 0; q < K2_NPOS; ++q) {
        a2[2 * q] = ffma2(x01[q], kn2[q], cn2[q]);                 /* -u */
        a2[2 * q + 1] = ffma2(x23[q], kn2[q], cn2[q]);
    }
    const f32x2 mone2 = pack2(-1.f, -1.f);
#pragma unroll
    for (int i = 0; i < 2 * K2_NPOS; ++i) {
        float a0, a1;
        unpack2(a2[i], a0, a1);
        f32x2 ne2;
        if constexpr (APOW >= 0) {                                  /* alpha = 2^APOW: no multiply (umi_device.cuh) */
            ne2 = pack2(neg_ueff_clamped_pow2<APOW>(a0), neg_ueff_clamped_pow2<APOW>(a1));
        } else {
            const f32x2 b2 = fmul2(a2[i], nalpha2);                /* alpha*u */
            float b0, b1;
            unpack2(b2, b0, b1);
            ne2 = pack2(neg_ueff_clamped(a0, b0), neg_ueff_clamped(a1, b1));
        }
        const f32x2 n2 = ffma2(ne2, ne2, mone2);                   /* -(1 - e^2) <= 0 */
        w2[i] = fmul2(n2, n2);                                     /* Eq. 3 */
    }
#pragma unroll
    for (int q = 0; q < K2_NPOS; ++q) {
        S2[q] = fadd2(S2[q], fadd2(w2[2 * q], w2[2 * q + 1]));
        /* sum w x on the sample pairs themselves (shared by the 4 positions in an interior group), so that u need not stay live */
        R2[q] = ffma2(w2[2 * q], x01[q], R2[q]);
        R2[q] = ffma2(w2[2 * q + 1], x23[q], R2[q]);
    }
}

/* Phase 2 with n+ known (the median kernel counts it exactly, on the sorted keys): Eq. 1 is a sum of squares only.
   d = x - med on sample pairs (FADD2), max(d, 0) as a signed-integer maximum on the ALU pipe, ss += d*d (FFMA2):
   two FMA-pipe lane-operations and one ALU instruction per sample. */
__device__ __forceinline__ void eval_scale_group(const f32x2 (&x01)[K2_NPOS], const f32x2 (&x23)[K2_NPOS],
                                                 const f32x2 (&nmed2)[K2_NPOS], f32x2 (&ss2)[K2_NPOS])
{
#pragma unroll
    for (int q = 0; q < K2_NPOS; ++q) {
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            const f32x2 d2 = fadd2(hh ? x23[q] : x01[q], nmed2[q]);
            float d0, d1;
            unpack2(d2, d0, d1);
            const f32x2 p2 = pack2(__int_as_float(max(__float_as_int(d0), 0)),
                                   __int_as_float(max(__float_as_int(d1), 0)));
            ss2[q] = ffma2(p2, p2, ss2[q]);
        }
    }
}

} // namespace

/* MODE 0: the paper's path.  MODE 1: sibling estimators with bisquare weights (scale from a buffer
   and / or written out).  MODE 2: the same with Welsch weights. */
/* SPLIT > 1 (small batches, where the grid would not fill the GPU): SPLIT adjacent lanes share the 4
   positions, each taking every SPLIT-th 128-bit group of the windows; the partial sums are combined
   with xor shuffles after every pass.  A warp tile then holds K2_WARP_TILE / SPLIT positions and a thread's serial
   chain is SPLIT times shorter.  SPLIT = 1 is the throughput configuration.
   APOW >= 0: the launch has alpha = 2^APOW and the interior loop forms alpha*u without a multiply;
   warps in which -u could overflow run all their groups through the scalar edge loop instead. */
template <int MODE, int SPLIT, int APOW>
__global__ void __launch_bounds__(K2_THREADS, (APOW >= 0 && SPLIT == 1) ? UMI_K2_MIN_CTAS_POW2 : UMI_K2_MIN_CTAS)
umi_reweight_kernel(ReweightParams prm)
{
    constexpr int TILE = K2_WARP_TILE / SPLIT;          /* positions per warp tile */
    extern __shared__ __align__(16) unsigned char smem_raw[];

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int pt = lane / SPLIT;                        /* which 4 positions of the tile */
    const int sl = lane % SPLIT;                        /* which slice of their windows */
    const int W = prm.W;
    const int h = (W - 1) >> 1;
    const int hal = (h + 3) & ~3;
    const int delta = hal - h;
    const int G = (3 + delta + 2 * h) / 4 + 1;          /* float4 groups per thread */
    const int nx = TILE + 4 * G;                        /* staged floats per warp (a multiple of 4) */
    const int g_lo = (3 + delta + 3) >> 2;              /* first group fully inside all 4 windows */
    const int g_hi = (delta + 2 * h - 3) >= 0 ? ((delta + 2 * h - 3) >> 2) : -1;   /* last such group */
    /* first interior group of this lane's slice: the smallest g >= g_lo with g = sl (mod SPLIT) */
    const int g_first = (SPLIT == 1) ? g_lo : g_lo + ((sl - g_lo % SPLIT) + SPLIT) % SPLIT;
    const float nalpha = -prm.alpha;
    const float qnan = __int_as_float(0x7FC00000);
    float* xs = reinterpret_cast<float*>(smem_raw) + warp * nx;     /* this warp's slice */
    const bool vec = (prm.N & 3) == 0 && (reinterpret_cast<uintptr_t>(prm.flux) & 15) == 0 &&
                     (reinterpret_cast<uintptr_t>(prm.time) & 15) == 0;

    for (int64_t bid = (int64_t)blockIdx.x * K2_WARPS + warp; bid < prm.n_blocks; bid += (int64_t)gridDim.x * K2_WARPS) {
        const int64_t star = bid / prm.tiles_per_star;
        const int64_t tile = bid - star * prm.tiles_per_star;
        const int64_t j0 = tile * TILE;
        const int64_t jbase = j0 - hal;                 /* cadence of staged index 0 */
        const float* frow = prm.flux + star * prm.N;
        const double* trow = prm.time ? prm.time + star * prm.N : nullptr;
        float* otile = prm.out + star * prm.N + j0;          /* the tile's TILE positions of the output row */
        const int nrow = (int)((prm.N - j0 < TILE) ? prm.N - j0 : TILE);   /* positions of the tile inside the row */

        /* stage the union, NaN marks invalid; tile min / max of the valid samples.  jbase is a multiple of 4, so
           when the rows are 16-byte aligned (vec: N % 4 == 0 and aligned base pointers) a lane moves four samples
           with one 128-bit load (two for an fp64 time), all of a round's loads in flight before the first use;
           otherwise one 32-bit load per sample, four in flight */
        float tmin = INFINITY, tmax = -INFINITY;
        if (vec) {
            for (int u = 4 * lane; u < nx; u += 128) {
                const int64_t j = jbase + u;
                float4 v = make_float4(qnan, qnan, qnan, qnan);
                if (j >= 0 && j < prm.N) {                  /* a group of 4 lies entirely inside or outside the row */
                    v = __ldg(reinterpret_cast<const float4*>(frow + j));
                    bool t0 = true, t1 = true, t2 = true, t3 = true;
                    if (trow != nullptr) {
                        const double2 ta = __ldg(reinterpret_cast<const double2*>(trow + j));
                        const double2 tb = __ldg(reinterpret_cast<const double2*>(trow + j + 2));
                        t0 = finite_f64(ta.x); t1 = finite_f64(ta.y); t2 = finite_f64(tb.x); t3 = finite_f64(tb.y);
                    }
                    v.x = (t0 && finite_f32(v.x)) ? v.x : qnan;
                    v.y = (t1 && finite_f32(v.y)) ? v.y : qnan;
                    v.z = (t2 && finite_f32(v.z)) ? v.z : qnan;
                    v.w = (t3 && finite_f32(v.w)) ? v.w : qnan;
                    tmin = fminf(tmin, fminf(fminf(v.x, v.y), fminf(v.z, v.w)));     /* fminf / fmaxf skip NaN */
                    tmax = fmaxf(tmax, fmaxf(fmaxf(v.x, v.y), fmaxf(v.z, v.w)));
                }
                *reinterpret_cast<float4*>(xs + u) = v;
            }
        } else {
            for (int u0 = 0; u0 < nx; u0 += 128) {
                float xv[4];
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int u = u0 + 32 * r + lane;
                    float x = 0.f;
                    const bool ok = u < nx && load_sample(trow, frow, prm.N, jbase + u, x);
                    xv[r] = ok ? x : qnan;
                }
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int u = u0 + 32 * r + lane;
                    tmin = fminf(tmin, xv[r]);
                    tmax = fmaxf(tmax, xv[r]);
                    if (u < nx) xs[u] = xv[r];
                }
            }
        }
        __syncwarp();
        pdl_wait_for_primary();                             /* the median kernel's words are complete and visible from here on */

        /* per-position state: 4 consecutive positions, local index 4*pt + q.  The median: read from the staged
           window at the offset the median kernel handed over (with n+), or an fp32 value (sibling estimators) */
        float mu[K2_NPOS], kk[K2_NPOS], cs[K2_NPOS];
        float nplus[K2_NPOS] = {0.f, 0.f, 0.f, 0.f};
        bool act[K2_NPOS];
        bool any_act = false;
        unsigned has_med = 0u;                              /* bit q: position q has a median, i.e. a trend */
        float rabs = INFINITY, rval = 0.f;                  /* the tile's median of smallest magnitude: the reference */
#pragma unroll
        for (int q = 0; q < K2_NPOS; ++q) {
            const int jl = 4 * pt + q;                      /* position inside the tile (32-bit from here on) */
            float med = qnan;
            if (jl < nrow) {
                if (MODE == 0 || prm.packed) {
                    const uint32_t word = reinterpret_cast<const uint32_t*>(otile)[jl];
                    if (word != HANDOVER_NONE) {
                        med = xs[jl + delta + (int)(word & 0xFFFFu)];   /* window of jl = staged [jl + delta, jl + delta + 2h] */
                        nplus[q] = (float)(word >> 16);
                    }
                } else {
                    med = otile[jl];
                }
            }
            act[q] = (med == med);
            has_med |= act[q] ? (1u << q) : 0u;
            any_act = any_act || act[q];
            mu[q] = act[q] ? med : 0.f;
            if (act[q] && fabsf(med) < rabs) { rabs = fabsf(med); rval = med; }
            kk[q] = 0.f;
            cs[q] = 0.f;
            if constexpr (MODE != 0) {                              /* no trend, no scale */
                if (prm.scale_in == nullptr && prm.scale_out != nullptr && jl < nrow && !act[q] && sl == 0)
                    prm.scale_out[star * prm.N + j0 + jl] = qnan;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            tmin = fminf(tmin, __shfl_xor_sync(0xFFFFFFFFu, tmin, o));
            tmax = fmaxf(tmax, __shfl_xor_sync(0xFFFFFFFFu, tmax, o));
            const float oabs = __shfl_xor_sync(0xFFFFFFFFu, rabs, o), oval = __shfl_xor_sync(0xFFFFFFFFu, rval, o);
            if (oabs < rabs || (oabs == rabs && oval < rval)) { rabs = oabs; rval = oval; }   /* (every lane ends with the same pick) */
        }
        /* sentinel: alpha*(mu - x)/(c s) >= 2 for every window of the tile, since
           mu >= tmin and s <= 0.6745 (tmax - tmin)  ("Sentinel") */
        float sent = 0.f;
        if (tmin <= tmax) {
            if constexpr (MODE == 0)
                sent = tmin - (2.f * SCALE_CONST) * prm.c_over_alpha * (tmax - tmin);
            else   /* s <= tmax - tmin for either scale; Welsch needs |u_eff| >= 16 for an exact 0 */
                sent = tmin - (MODE == 2 ? 24.f : 2.f) * prm.c_over_alpha * (tmax - tmin);
            sent = fmaxf(sent, -3.0e38f);
        }
        /* Everything below works on samples centred on ONE OF THE TILE'S MEDIANS, the one of smallest magnitude: Eq. 4 is
           then mu' = sum(w x') / sum(w) with |x'| small for every sample that can carry weight, i.e. exact to fp32 without
           a separate sum of w*u.  A median is robust: a wild sample (a fill value, a glitch of any size) cannot move it,
           keeps its own magnitude in x' and leaves the precision of the others alone.  And the smallest one is safe when
           the tile's medians themselves disagree (the edge of a run of unmasked fill values: medians of -9999 next to
           medians of 1): |x_ref| <= |median of p| for every position p, so the samples near p's median lose at most one
           bit to the centring, whatever the other positions of the tile look like. */
        const float xref = (rabs < INFINITY) ? rval : 0.f;
        const float xsent = sent - xref;                    /* the sentinel as staged */
        const float xabs = (tmin <= tmax) ? fmaxf(fabsf(xsent), fabsf(tmax - xref)) : 0.f;         /* max |x'| staged */
        __syncwarp();                                       /* every lane has read its medians from xs */
        for (int u = lane; u < nx; u += 32) {
            const float x = xs[u];
            xs[u] = (x != x) ? xsent : x - xref;
        }
#pragma unroll
        for (int q = 0; q < K2_NPOS; ++q) mu[q] = act[q] ? mu[q] - xref : 0.f;
        __syncwarp();

        const float4* xs4 = reinterpret_cast<const float4*>(xs) + pt;

        if (__any_sync(0xFFFFFFFFu, any_act)) {
            /* Edge groups hold samples that belong to some but not all of the thread's 4 windows.  The throughput variant
               (SPLIT = 1) runs its two or three of them one (sample, position) at a time, predicated.  The split-window
               variant, where a lane has ~1/SPLIT of the groups and the edge groups weigh SPLIT times more, runs them through
               the same packed arithmetic as the interior groups on MASKED samples: position q sees the (centred) sentinel
               in place of a sample outside its window -- never above a median, weight exactly 0.  There the lane's groups
               g = sl, sl + SPLIT, ... < G fall into three runs: [sl, g_first) low edge groups; [g_first, g_tail) interior
               groups, a multiple of 8 of them, through the unrolled loop; [g_tail, G) the rest -- up to 7 interior groups and
               the high edge groups -- through the same rolled, masked loop as the low edge groups (one copy of its body). */
            constexpr int UNR = K2_UNROLL;
            int g_tail = g_first;
            if (g_first <= g_hi) g_tail += ((g_hi - g_first) / SPLIT + 1) / UNR * (UNR * SPLIT);
            const unsigned two_h = 2u * (unsigned)h;
            auto masked_group = [&](int g, f32x2 (&x01)[K2_NPOS], f32x2 (&x23)[K2_NPOS]) {
                const float4 v = xs4[g];
#pragma unroll
                for (int q = 0; q < K2_NPOS; ++q) {
                    const int o = 4 * g - delta - q;                    /* offset of v.x inside window q */
                    x01[q] = pack2((unsigned)o <= two_h ? v.x : xsent, (unsigned)(o + 1) <= two_h ? v.y : xsent);
                    x23[q] = pack2((unsigned)(o + 2) <= two_h ? v.z : xsent, (unsigned)(o + 3) <= two_h ? v.w : xsent);
                }
            };
            auto shared_group = [&](int g, f32x2 (&x01)[K2_NPOS], f32x2 (&x23)[K2_NPOS]) {
                const ulonglong2 v2 = reinterpret_cast<const ulonglong2*>(xs4)[g];
#pragma unroll
                for (int q = 0; q < K2_NPOS; ++q) { x01[q] = v2.x; x23[q] = v2.y; }
            };

            /* ---- Phase 2 (Eq. 1) ---- */
            float ss[K2_NPOS], cnt[K2_NPOS];
#pragma unroll
            for (int q = 0; q < K2_NPOS; ++q) { ss[q] = 0.f; cnt[q] = 0.f; }
            const bool given = (MODE != 0) && prm.scale_in != nullptr;
            if constexpr (MODE == 0) {                              /* n+ came with the median: a sum of squares is left */
                f32x2 nmed2[K2_NPOS], ss2[K2_NPOS], x01[K2_NPOS], x23[K2_NPOS];
#pragma unroll
                for (int q = 0; q < K2_NPOS; ++q) { nmed2[q] = pack2(-mu[q], -mu[q]); ss2[q] = pack2(0.f, 0.f); }
                if constexpr (SPLIT == 1) {
                    for (int g = 0; g < G; ++g) {                   /* edge groups, one (sample, position) at a time */
                        if (g == g_lo && g_hi >= g_lo) g = g_hi + 1;
                        if (g >= G) break;
                        const float4 v = xs4[g];
                        const float xv[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                        for (int q = 0; q < K2_NPOS; ++q)
#pragma unroll
                            for (int r = 0; r < 4; ++r)
                                if ((unsigned)(4 * g + r - delta - q) <= two_h) eval_scale(xv[r], mu[q], ss[q], cnt[q]);
                    }
#pragma unroll 8
                    for (int g = g_lo; g <= g_hi; ++g) {
                        shared_group(g, x01, x23);
                        eval_scale_group(x01, x23, nmed2, ss2);
                    }
                } else {
                    for (int g = sl; g < G; g += SPLIT) {
                        if (g == g_first) g = g_tail;
                        if (g >= G) break;
                        masked_group(g, x01, x23);
                        eval_scale_group(x01, x23, nmed2, ss2);
                    }
                    for (int g0 = g_first; g0 < g_tail; g0 += UNR * SPLIT) {
#pragma unroll
                        for (int j = 0; j < UNR; ++j) {
                            shared_group(g0 + j * SPLIT, x01, x23);
                            eval_scale_group(x01, x23, nmed2, ss2);
                        }
                    }
                }
#pragma unroll
                for (int q = 0; q < K2_NPOS; ++q) {
                    float s0, s1;
                    unpack2(ss2[q], s0, s1);
                    ss[q] += s0 + s1;
                }
            } else {                                                /* sibling estimators: count and sum, one sample at a time */
                for (int g = sl; g < (given ? 0 : G); g += SPLIT) {
                    const float4 v = xs4[g];
                    const float xv[4] = {v.x, v.y, v.z, v.w};
                    if (g >= g_lo && g <= g_hi) {                   /* interior: every sample in all 4 windows */
#pragma unroll
                        for (int q = 0; q < K2_NPOS; ++q)
#pragma unroll
                            for (int r = 0; r < 4; ++r) eval_scale(xv[r], mu[q], ss[q], cnt[q]);
                    } else {
#pragma unroll
                        for (int q = 0; q < K2_NPOS; ++q)
#pragma unroll
                            for (int r = 0; r < 4; ++r)
                                if ((unsigned)(4 * g + r - delta - q) <= two_h) eval_scale(xv[r], mu[q], ss[q], cnt[q]);
                    }
                }
            }
            if constexpr (SPLIT > 1) {
#pragma unroll
                for (int q = 0; q < K2_NPOS; ++q)
#pragma unroll
                    for (int o = SPLIT / 2; o > 0; o >>= 1) {
                        ss[q] += __shfl_xor_sync(0xFFFFFFFFu, ss[q], o);
                        if constexpr (MODE != 0) cnt[q] += __shfl_xor_sync(0xFFFFFFFFu, cnt[q], o);
                    }
            }
            if constexpr (MODE == 0) {
#pragma unroll
                for (int q = 0; q < K2_NPOS; ++q) cnt[q] = nplus[q];
            }
#pragma unroll
            for (int q = 0; q < K2_NPOS; ++q) {
                bool on = act[q] && cnt[q] > 0.f;                   /* (R8) */
                float s = 0.f;
                if (on) {
                    s = SCALE_CONST * sqrtf(ss[q] / cnt[q]);
                    on = s > 0.f;
                }
                if constexpr (MODE != 0) {
                    const int jl = 4 * pt + q;
                    if (given) {                                    /* the MAD from the selection kernel */
                        s = (act[q] && jl < nrow) ? prm.scale_in[star * prm.N + j0 + jl] : 0.f;
                        on = act[q] && s > 0.f;
                    } else if (prm.scale_out != nullptr && jl < nrow && act[q] && sl == 0) {
                        prm.scale_out[star * prm.N + j0 + jl] = s;
                    }
                }
                act[q] = on;
                cs[q] = on ? prm.c * s : 0.f;
                kk[q] = on ? 1.f / cs[q] : 0.f;
            }

            /* the packed loops form -u = k (mu' - x') without a guard, and the alpha = 2^APOW form of alpha*u would
               wrap an overflowed -u to a small value: warps in which it could overflow (|x'|, |mu'| <= xabs; never
               seen on real data) run every group through the scalar loop, which multiplies and predicates */
            bool risky = false;
#pragma unroll
            for (int q = 0; q < K2_NPOS; ++q) risky = risky || !(kk[q] * xabs < 1.2676506e30f);   /* 2^100 */
            risky = __any_sync(0xFFFFFFFFu, risky);
            /* ---- Phase 3 (Eq. 2-4), s held fixed (R9), exactly n_iter passes (R10) ---- */
            for (int it = 0; it < prm.n_iter; ++it) {
                float S[K2_NPOS], R[K2_NPOS], c0[K2_NPOS];
#pragma unroll
                for (int q = 0; q < K2_NPOS; ++q) { S[q] = 0.f; R[q] = 0.f; c0[q] = -mu[q] * kk[q]; }
                f32x2 S2[K2_NPOS], R2[K2_NPOS], kn2[K2_NPOS], cn2[K2_NPOS], x01[K2_NPOS], x23[K2_NPOS];
                const f32x2 nalpha2 = pack2(nalpha, nalpha);
#pragma unroll
                for (int q = 0; q < K2_NPOS; ++q) {
                    S2[q] = pack2(0.f, 0.f);
                    R2[q] = pack2(0.f, 0.f);
                    kn2[q] = pack2(-kk[q], -kk[q]);                 /* exact negations: u' = -u bit for bit */
                    cn2[q] = pack2(-c0[q], -c0[q]);
                }
                const bool scalar_all = risky;
                if (SPLIT == 1 || scalar_all) {
                    /* one (sample, position) at a time, predicated: every group of a `risky` warp; in the
                       throughput variant also the two or three edge groups (measured against the masked form
                       below: 6.95 vs 7.00 ms at W = 361, 53.1 vs 54.9 at W = 217, 46.9 vs 47.3 at W = 2161 -- a
                       second packed loop body costs more in instruction cache than it saves in issue slots) */
                    for (int g = sl; g < G; g += SPLIT) {
                        if (!scalar_all && g >= g_lo && g <= g_hi) {
                            g = g_hi;                               /* (SPLIT == 1 here) */
                            continue;
                        }
                        const float4 v = xs4[g];
                        const float xv[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                        for (int q = 0; q < K2_NPOS; ++q)
#pragma unroll
                            for (int r = 0; r < 4; ++r)
                                if ((unsigned)(4 * g + r - delta - q) <= two_h) {
                                    if constexpr (MODE == 2) eval_welsch(xv[r], kk[q], c0[q], nalpha, S[q], R[q]);
                                    else eval_weight(xv[r], kk[q], c0[q], nalpha, S[q], R[q]);
                                }
                    }
                }
                if constexpr (MODE == 2) {
                    if (!scalar_all) {                              /* Welsch: MUFU-bound, one sample at a time */
#pragma unroll 2
                        for (int g = g_lo; g <= g_hi; ++g) {
                            const float4 v = xs4[g];
                            const float xv[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                            for (int q = 0; q < K2_NPOS; ++q)
#pragma unroll
                                for (int r = 0; r < 4; ++r) eval_welsch(xv[r], kk[q], c0[q], nalpha, S[q], R[q]);
                        }
                    }
                } else {
                    if (!scalar_all) {
                        if constexpr (SPLIT == 1) {
#pragma unroll K2_UNROLL
                            for (int g = g_lo; g <= g_hi; ++g) {       /* interior groups: every sample belongs to all 4 windows */
                                shared_group(g, x01, x23);
                                eval_weight_group<APOW>(x01, x23, kn2, cn2, nalpha2, S2, R2);
                            }
                        } else {
                            /* split-window variant: a lane has ~1/SPLIT of the groups, so the edge groups weigh SPLIT
                               times more: masked, packed, in the rolled loop that also takes what the unrolled one
                               leaves over (config 1: 30.7 -> 26.6 us) */
                            for (int g = sl; g < G; g += SPLIT) {
                                if (g == g_first) g = g_tail;
                                if (g >= G) break;
                                masked_group(g, x01, x23);
                                eval_weight_group<APOW>(x01, x23, kn2, cn2, nalpha2, S2, R2);
                            }
                            for (int g0 = g_first; g0 < g_tail; g0 += UNR * SPLIT) {
#pragma unroll
                                for (int j = 0; j < UNR; ++j) {
                                    shared_group(g0 + j * SPLIT, x01, x23);
                                    eval_weight_group<APOW>(x01, x23, kn2, cn2, nalpha2, S2, R2);
                                }
                            }
                        }
#pragma unroll
                        for (int q = 0; q < K2_NPOS; ++q) {
                            float s0, s1, r0, r1;
                            unpack2(S2[q], s0, s1);
                            unpack2(R2[q], r0, r1);
                            S[q] += s0 + s1;
                            R[q] += r0 + r1;
                        }
                    }
                }
#pragma unroll
                for (int q = 0; q < K2_NPOS; ++q) {
                    if constexpr (SPLIT > 1) {
#pragma unroll
                        for (int o = SPLIT / 2; o > 0; o >>= 1) {
                            S[q] += __shfl_xor_sync(0xFFFFFFFFu, S[q], o);
                            R[q] += __shfl_xor_sync(0xFFFFFFFFu, R[q], o);
                        }
                    }
                    if (act[q] && S[q] > 0.f) mu[q] = R[q] / S[q];                       /* Eq. 4; (R11) */
                }
            }
        }

        /* the trend; with n_iter = 0 (sibling estimators asked for the scale only) `out` keeps the median
           the selection kernel wrote, bit for bit */
        float* flrow = prm.flat != nullptr ? prm.flat + star * prm.N + j0 : nullptr;
#pragma unroll
        for (int q = 0; q < K2_NPOS; ++q) {
            const int jl = 4 * pt + q;
            if (jl < nrow && sl == 0) {
                const bool has = (has_med >> q) & 1u;
                float tr = mu[q] + xref;
                if (MODE != 0 && prm.n_iter == 0) tr = otile[jl];
                else otile[jl] = has ? tr : qnan;
                if (flrow != nullptr)                               /* PAPER.md:155 normalisation */
                    flrow[jl] = has ? __ldg(frow + j0 + jl) / tr : qnan;
            }
        }
        __syncwarp();                                       /* the slice is free for the next tile */
    }
}

cudaError_t launch_reweight(const ReweightParams& prm, bool family, unsigned grid, size_t smem, cudaStream_t stream)
{
    const int ap = alpha_pow2(prm.alpha);
    void (*k2)(ReweightParams) = nullptr;
    if (!family && prm.split == K2_SPLIT) k2 = (ap == 1) ? umi_reweight_kernel<0, K2_SPLIT, 1> : umi_reweight_kernel<0, K2_SPLIT, -1>;
    else if (!family) k2 = (ap == 0) ? umi_reweight_kernel<0, 1, 0> : (ap == 1) ? umi_reweight_kernel<0, 1, 1>
                         : (ap == 2) ? umi_reweight_kernel<0, 1, 2> : umi_reweight_kernel<0, 1, -1>;
    else k2 = (prm.weight_kind == WEIGHT_WELSCH) ? umi_reweight_kernel<2, 1, -1> : umi_reweight_kernel<1, 1, -1>;
    if (smem > 48 * 1024) {               /* W > ~2900: four warp slices of W + 131 floats pass the default limit */
        const cudaError_t e = cudaFuncSetAttribute(k2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    /* programmatic dependent launch behind the median kernel (umi_device.cuh): the prologue of this grid --
       launch, staging of the samples -- overlaps the tail of that one */
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(K2_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, k2, prm);
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}

} // namespace umi
