/*
 * umi_reweight_tc.cu -- Phase 2 + Phase 3 (Eq. 1-4) with the two weighted sums of
 * Eq. 4 on the 5th-generation tensor cores (tcgen05, accumulators in TMEM).
 *
 * Why: the weights w(p, j) of Eq. 2-3 depend on the position's own mu and s, so they are computed on
 * the CUDA cores exactly as in umi_reweight.cu (u = x k + c0, e = max(u, -alpha u),
 * w = max(1 - e^2, 0)^2: 4 FMA-pipe + 2 ALU-pipe operations per (sample, position)).  But once a
 * weight exists, Eq. 4's   sum_j w(p, j) [1, x_j]   is a dense (banded) contraction: rows =
 * positions, K = samples, two useful columns.  On the FMA pipe it costs 2 of the 6 lane-operations
 * of an evaluation and the kernel is FMA-pipe bound (dropping one of them alone took umi_reweight
 * from 8.78 to 6.90 ms on config 2).  Here a thread writes its row of weights into TMEM
 * (tcgen05.st, 16 per instruction) and one thread issues  D[128 x 16] += A[128 x 8] B[8 x 16]
 * (kind::tf32, A from TMEM, B from shared memory) per 8 samples.
 *
 * Numerics.  tf32 operands, fp32 accumulation.  The weight is TRUNCATED to tf32 by the tensor core
 * (10 mantissa bits, measured: the result matches truncation, not rounding) -- the same truncated
 * weight multiplies every column, so   mu <- sum(w~ x) / sum(w~)   is an exactly consistent weighted
 * mean with weights perturbed by < 2^-10 relative (one-sided), which moves mu by
 * <~ 5e-4 * |weighted mean of (x - mu) over a random sign| ~ 1e-8 of the flux.  The samples are centred
 * on a per-tile reference x_ref and split exactly into three tf32 terms x' = xh + xm + xl (columns
 * 1-3 of B; column 0 is 1), so no sample bit is lost.  Everything (mu, median) is carried as an
 * offset from x_ref.
 *
 * CTA = 128 producer threads (one position = one TMEM lane each) + 1 issuer warp; tile = 128
 * positions; the windows of a tile span NCH chunks of 16 samples.  Ring of 3 TMEM stages
 * (16 columns each) + 16 accumulator columns = 64 TMEM columns per CTA.
 *   producers: wait free[stage] -> 16 weights -> tcgen05.st -> wait::st -> arrive full[stage]
 *   issuer:    wait full[stage] -> 2 x tcgen05.mma (K = 8) -> tcgen05.commit -> free[stage]
 *   end of pass: tcgen05.commit -> done; producers tcgen05.ld their row (S, T1, T2, T3),
 *                mu' = (T1 + T2 + T3) / S  (Eq. 4), arrive dfree.
 * Nothing here is shared with oracle/.
 */
#include "umi_device.cuh"

namespace umi {

namespace {

constexpr int TC_POS = 128;                 /* positions (= TMEM lanes) per CTA */
constexpr int TC_THREADS = TC_POS + 32;     /* + the issuer warp */
constexpr int TC_CHUNK = 16;                /* samples per unit of work (one tcgen05.st) */
constexpr int TC_STAGE = 2 * TC_CHUNK;      /* samples per hand-over to the tensor core */
constexpr int TC_COLS = 64;                 /* TMEM columns: 32 (A stage) + 16 (D), rounded up to a power of two */
constexpr uint32_t TC_DCOL = TC_STAGE;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* b, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
/* Wait for the phase with the given parity.  try_wait suspends the thread in hardware for up to the
   hinted time, so the loop rarely iterates; it is bounded so that a protocol error traps instead of
   hanging the GPU. */
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity)
{
    const uint32_t addr = smem_u32(b);
    uint32_t done = 0;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(done) : "r"(addr), "r"(parity) : "memory");
    if (done) return;
    for (int spins = 0; !done; ++spins) {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(done) : "r"(addr), "r"(parity), "r"(100000u) : "memory");
        if (spins > (1 << 20)) __trap();
    }
}

/* K-major, no swizzle: core matrix = 8 rows x 16 bytes; LBO = stride between core matrices along K,
   SBO = stride between 8-row groups along N (0: rows 8-15 alias rows 0-7, their columns are ignored). */
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
    d |= (uint64_t)((lbo >> 4) & 0x3FFF) << 16;
    d |= (uint64_t)((sbo >> 4) & 0x3FFF) << 32;
    d |= (uint64_t)1 << 46;                 /* descriptor version of sm_100 */
    return d;
}

/* instruction descriptor: D = f32, A = B = tf32, both K-major, N = 16, M = 128 */
constexpr uint32_t TC_IDESC = (1u << 4) | (2u << 7) | (2u << 10) | ((16u >> 3) << 17) | ((128u >> 4) << 24);

__device__ __forceinline__ void tmem_st16(uint32_t taddr, const float (&w)[TC_CHUNK])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
        ::"r"(taddr), "f"(w[0]), "f"(w[1]), "f"(w[2]), "f"(w[3]), "f"(w[4]), "f"(w[5]), "f"(w[6]), "f"(w[7]),
        "f"(w[8]), "f"(w[9]), "f"(w[10]), "f"(w[11]), "f"(w[12]), "f"(w[13]), "f"(w[14]), "f"(w[15])
        : "memory");
}

__device__ __forceinline__ float tf32_trunc(float x) { return __uint_as_float(__float_as_uint(x) & 0xFFFFE000u); }


enum ChunkKind { CHUNK_ZERO = 0, CHUNK_LEFT = 1, CHUNK_RIGHT = 2, CHUNK_INTERIOR = 3 };

/* 16 weights of one position for the samples of chunk c (Eq. 2-3).  LEFT / RIGHT chunks lie across the
   start / the end of some window of the warp: samples outside this thread's window [tid, tid + 2h] get
   weight 0 through a 0/1 factor built on the FMA pipe (sat of a difference), not a compare + select. */
template <int KIND>
__device__ __forceinline__ void chunk_weights(const float4* xs4, int c, int tid, int h2, f32x2 k2, f32x2 c02, f32x2 na2,
                                              float (&w)[TC_CHUNK])
{
    if constexpr (KIND == CHUNK_ZERO) {
#pragma unroll
        for (int i = 0; i < TC_CHUNK; ++i) w[i] = 0.f;
    } else {
#pragma unroll
        for (int g = 0; g < 4; ++g) {
            const ulonglong2 v2 = reinterpret_cast<const ulonglong2*>(xs4)[4 * c + g];
#pragma unroll
            for (int hlf = 0; hlf < 2; ++hlf) {
                const f32x2 x2 = hlf ? v2.y : v2.x;
                const f32x2 a2 = ffma2(x2, k2, c02);                /* u */
                const f32x2 b2 = fmul2(a2, na2);                    /* -alpha u */
                float a0, a1, b0, b1;
                unpack2(a2, a0, a1);
                unpack2(b2, b0, b1);
                /* the FMA pipe has room here (no accumulation on it): the clamp of Eq. 3 (R12) is the .SAT of a
                   scalar FFMA, which leaves one FMNMX per evaluation on the half-rate ALU pipe */
                const float e0 = fmaxf(a0, b0), e1 = fmaxf(a1, b1);
                const f32x2 t2 = pack2(__saturatef(fmaf(-e0, e0, 1.f)), __saturatef(fmaf(-e1, e1, 1.f)));
                float w0, w1;
                unpack2(fmul2(t2, t2), w0, w1);
                w[4 * g + 2 * hlf] = w0;
                w[4 * g + 2 * hlf + 1] = w1;
            }
        }
        if constexpr (KIND == CHUNK_LEFT) {
            const float first = (float)(tid - TC_CHUNK * c);        /* element i is inside the window iff i >= first */
#pragma unroll
            for (int i = 0; i < TC_CHUNK; ++i) w[i] *= __saturatef((float)(i + 1) - first);
        }
        if constexpr (KIND == CHUNK_RIGHT) {
            const float last = (float)(tid + h2 - TC_CHUNK * c);    /* ... iff i <= last */
#pragma unroll
            for (int i = 0; i < TC_CHUNK; ++i) w[i] *= __saturatef(last - (float)(i - 1));
        }
    }
}

/* Phase 2 (Eq. 1) on one chunk */
template <int KIND>
__device__ __forceinline__ void chunk_scale(const float4* xs4, int c, int tid, int h2, float med, float& ss, float& cnt)
{
    float xv[TC_CHUNK];
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        const float4 v = xs4[4 * c + g];
        xv[4 * g] = v.x; xv[4 * g + 1] = v.y; xv[4 * g + 2] = v.z; xv[4 * g + 3] = v.w;
    }
    const unsigned first = (unsigned)(tid - TC_CHUNK * c);
#pragma unroll
    for (int i = 0; i < TC_CHUNK; ++i) {
        const float d = xv[i] - med;
        bool take = d > 0.f;
        if constexpr (KIND != CHUNK_INTERIOR) take = take && ((unsigned)i - first <= (unsigned)h2);
        if (take) { ss = fmaf(d, d, ss); cnt += 1.f; }
    }
}

} // namespace

#ifndef UMI_TC_MIN_CTAS
#define UMI_TC_MIN_CTAS 8
#endif
__global__ void __launch_bounds__(TC_THREADS, UMI_TC_MIN_CTAS)
umi_reweight_tc_kernel(ReweightParams prm, int nch)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* bm = reinterpret_cast<float*>(smem_raw);                 /* B: [nch][2 K-blocks][2 K-cores][8 rows][4] */
    float* xs = bm + (size_t)nch * 128;                             /* [16 nch] centred samples, sentinel where invalid */
    __shared__ __align__(8) uint64_t bar_full, bar_free, bar_done, bar_dfree;
    __shared__ uint32_t s_tmem;
    __shared__ float s_red[2 * (TC_POS / 32)];
    __shared__ float s_ref;

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const int W = prm.W;
    const int h = (W - 1) >> 1;
    const int nx = TC_CHUNK * nch;                                  /* >= TC_POS + 2h */
    const float qnan = __int_as_float(0x7FC00000);

    const int64_t bid = blockIdx.x;
    const int64_t star = bid / prm.tiles_per_star;
    const int64_t tile = bid - star * prm.tiles_per_star;
    const int64_t j0 = tile * TC_POS;
    const int64_t jbase = j0 - h;                                   /* cadence of staged index 0 */
    const float* frow = prm.flux + star * prm.N;
    const double* trow = prm.time ? prm.time + star * prm.N : nullptr;
    float* orow = prm.out + star * prm.N;

    if (tid == 0) {
        mbar_init(&bar_full, TC_POS / 32);
        mbar_init(&bar_free, 1);
        mbar_init(&bar_done, 1);
        mbar_init(&bar_dfree, TC_POS / 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == TC_POS / 32) {                                      /* the issuer warp owns the TMEM allocation */
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "n"(TC_COLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }

    /* stage the union; tile min / max of the valid samples; reference = median at the tile centre */
    float tmin = INFINITY, tmax = -INFINITY;
    for (int u = tid; u < nx; u += TC_THREADS) {
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
    if (lane == 0 && warp < TC_POS / 32) { s_red[warp * 2] = tmin; s_red[warp * 2 + 1] = tmax; }
    if (warp == TC_POS / 32 && lane == 0) { bm[0] = tmin; bm[1] = tmax; }     /* 5th warp's share, scratch */
    if (tid == 0) {
        const int64_t jc = j0 + TC_POS / 2;
        const float mc = (jc < prm.N) ? orow[jc] : qnan;
        s_ref = mc;                                                 /* may be NaN: fixed below */
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem = s_tmem;
    tmin = fminf(bm[0], tmin);
    tmax = fmaxf(bm[1], tmax);
#pragma unroll
    for (int w = 0; w < TC_POS / 32; ++w) {
        tmin = fminf(tmin, s_red[2 * w]);
        tmax = fmaxf(tmax, s_red[2 * w + 1]);
    }
    float xref = s_ref;
    if (!(xref == xref)) xref = (tmin <= tmax) ? 0.5f * tmin + 0.5f * tmax : 0.f;
    /* sentinel: alpha (mu - x)/(c s) >= 2 for every window of the tile ("Sentinel") */
    float sent = 0.f;
    if (tmin <= tmax) {
        sent = tmin - (2.f * SCALE_CONST) * prm.c_over_alpha * (tmax - tmin);
        sent = fmaxf(sent, -3.0e38f);
    }
    __syncthreads();                                                /* bm[0..1] scratch has been read */

    /* centre the samples; build B (column 0 = 1, columns 1-3 = exact tf32 split of x', rest 0) */
    for (int u = tid; u < nx; u += TC_THREADS) {
        const float x = xs[u];
        const bool ok = (x == x);
        const float xc = (ok ? x : sent) - xref;
        xs[u] = xc;
        const float xh = tf32_trunc(xc);
        const float xm = tf32_trunc(xc - xh);
        const float xl = tf32_trunc((xc - xh) - xm);
        /* element (row n, sample u): chunk u/16, K-block (u%16)/8, K-core (u%8)/4, e = u%4 */
        float* core = bm + (u >> 4) * 128 + ((u >> 3) & 1) * 64 + ((u >> 2) & 1) * 32 + (u & 3);
        core[0 * 4] = ok ? 1.f : 0.f;
        core[1 * 4] = ok ? xh : 0.f;
        core[2 * 4] = ok ? xm : 0.f;
        core[3 * 4] = ok ? xl : 0.f;
        core[4 * 4] = 0.f;
        core[5 * 4] = 0.f;
        core[6 * 4] = 0.f;
        core[7 * 4] = 0.f;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");    /* B is read by the tensor core (async proxy) */
    __syncthreads();

    if (warp == TC_POS / 32) {
        /* ---------------- issuer ---------------- */
        if (lane == 0) {
            const uint32_t bbase = smem_u32(bm);
            const int nst = nch / 2;
            const int span = (31 + 2 * h) / TC_STAGE;               /* warp w touches stages w .. w + span */
            uint32_t m = 0;
            for (int it = 0; it < prm.n_iter; ++it) {
                mbar_wait(&bar_dfree, (uint32_t)it & 1u);           /* D has been read and zeroed by every producer */
                for (int st = 0; st < nst; ++st, ++m) {
                    mbar_wait(&bar_full, m & 1u);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    /* rows of the warps whose windows do not reach this stage are left alone (they stored nothing) */
                    uint32_t dis[4];
#pragma unroll
                    for (int w = 0; w < 4; ++w) dis[w] = (st < w || st > w + span) ? 0xFFFFFFFFu : 0u;
#pragma unroll
                    for (int kb = 0; kb < 4; ++kb) {
                        const uint64_t bdesc = smem_desc(bbase + (uint32_t)(2 * st + (kb >> 1)) * 512u + (uint32_t)(kb & 1) * 256u, 128u, 0u);
                        const uint32_t a_t = tmem + kb * 8;
                        const uint32_t d_t = tmem + TC_DCOL;
                        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                                     "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, {%5, %6, %7, %8}, p;\n\t}"
                                     ::"r"(d_t), "r"(a_t), "l"(bdesc), "r"(TC_IDESC), "r"(1u),
                                       "r"(dis[0]), "r"(dis[1]), "r"(dis[2]), "r"(dis[3])
                                     : "memory");
                    }
                    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                                 ::"r"(smem_u32(&bar_free)) : "memory");
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                             ::"r"(smem_u32(&bar_done)) : "memory");
            }
        }
    } else {
        /* ---------------- producers: one position per thread ---------------- */
        const int64_t j = j0 + tid;
        const float med_raw = (j < prm.N) ? orow[j] : qnan;
        bool act = (med_raw == med_raw);
        const float med = act ? med_raw - xref : 0.f;
        float mu = med;
        const float4* xs4 = reinterpret_cast<const float4*>(xs);
        /* chunk classes for this warp: positions 32 warp .. 32 warp + 31, window of p = [p, p + 2h] */
        const int p_lo = 32 * warp, p_hi = 32 * warp + 31;
        const int c_first = p_lo / TC_CHUNK;                                    /* first chunk touching any window */
        const int c_last = (p_hi + 2 * h) / TC_CHUNK;                           /* last one */
        const int c_int_lo = (p_hi + TC_CHUNK - 1) / TC_CHUNK;                  /* first chunk inside all 32 windows */
        const int c_int_hi = (p_lo + 2 * h - (TC_CHUNK - 1)) >= 0 ? (p_lo + 2 * h - (TC_CHUNK - 1)) / TC_CHUNK : -1;

        /* ---- Phase 2 (Eq. 1) on the CUDA cores ---- */
        float ss = 0.f, cnt = 0.f;
        if (__any_sync(0xFFFFFFFFu, act)) {
            /* left edge, interior, right edge: three loops so that the interior carries no window test */
            int c = c_first;
            for (; c < c_int_lo && c <= c_last; ++c) chunk_scale<CHUNK_LEFT>(xs4, c, tid, 2 * h, med, ss, cnt);
            for (; c <= c_int_hi; ++c) chunk_scale<CHUNK_INTERIOR>(xs4, c, tid, 2 * h, med, ss, cnt);
            for (; c <= c_last; ++c) chunk_scale<CHUNK_LEFT>(xs4, c, tid, 2 * h, med, ss, cnt);
        }
        bool on = act && cnt > 0.f;                                             /* (R8) */
        float s = 0.f;
        if (on) {
            s = SCALE_CONST * sqrtf(ss / cnt);
            on = s > 0.f;
        }
        const float cs = on ? prm.c * s : 0.f;
        const float k = on ? 1.f / cs : 0.f;
        const f32x2 k2 = pack2(k, k), na2 = pack2(-prm.alpha, -prm.alpha);
        const uint32_t lane_base = tmem + ((uint32_t)(32 * warp) << 16);

        /* ---- Phase 3 (Eq. 2-4): weights here, the two sums on the tensor core ---- */
        const int nst = nch / 2;
        const int st_lo = warp, st_hi = warp + (31 + 2 * h) / TC_STAGE;         /* stages this warp's windows reach */
        auto zero_d = [&]() {
            asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%1,%1,%1};" ::"r"(lane_base + TC_DCOL), "r"(0u) : "memory");
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar_dfree);
        };
        /* 16 weights of chunk c, by class */
        auto weights = [&](int c, f32x2 c02, float (&w)[TC_CHUNK]) {
            if (c < c_first || c > c_last) chunk_weights<CHUNK_ZERO>(xs4, c, tid, 2 * h, k2, c02, na2, w);
            else if (c < c_int_lo) chunk_weights<CHUNK_LEFT>(xs4, c, tid, 2 * h, k2, c02, na2, w);
            else if (c <= c_int_hi) chunk_weights<CHUNK_INTERIOR>(xs4, c, tid, 2 * h, k2, c02, na2, w);
            else chunk_weights<CHUNK_RIGHT>(xs4, c, tid, 2 * h, k2, c02, na2, w);
        };
        zero_d();
        uint32_t m = 0;
        for (int it = 0; it < prm.n_iter; ++it) {
            const float c0 = -mu * k;
            const f32x2 c02 = pack2(c0, c0);
            for (int st = 0; st < nst; ++st, ++m) {
                /* the MMAs that read the previous stage are done (every warp waits, so that nobody runs ahead
                   of the barrier phase); warps outside the stage only keep the count */
                if (st >= st_lo && st <= st_hi) {
                    float w[TC_CHUNK];
                    weights(2 * st, c02, w);                                    /* overlaps the MMAs of the previous stage */
                    mbar_wait(&bar_free, (m & 1u) ^ 1u);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    tmem_st16(lane_base, w);
                    weights(2 * st + 1, c02, w);
                    tmem_st16(lane_base + TC_CHUNK, w);
                    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                    __syncwarp();
                } else {
                    mbar_wait(&bar_free, (m & 1u) ^ 1u);
                }
                if (lane == 0) mbar_arrive(&bar_full);
            }
            /* the pass is complete: read this position's row of D, then clear it for the next pass */
            mbar_wait(&bar_done, (uint32_t)it & 1u);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            float S, t1, t2, t3;
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
                         : "=f"(S), "=f"(t1), "=f"(t2), "=f"(t3)
                         : "r"(lane_base + TC_DCOL)
                         : "memory");
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (it + 1 < prm.n_iter) zero_d();
            if (on && S > 0.f) mu = ((t3 + t2) + t1) / S;                       /* Eq. 4 in centred coordinates; (R11) */
        }
        if (j < prm.N && act) {
            const float trend = mu + xref;
            orow[j] = trend;
            if (prm.flat != nullptr) prm.flat[star * prm.N + j] = __ldg(frow + j) / trend;
        } else if (j < prm.N && prm.flat != nullptr) {
            prm.flat[star * prm.N + j] = qnan;
        }
    }

    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == TC_POS / 32) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TC_COLS));
    }
}

/* chunks of 16 samples spanned by the windows of a 128-position tile */
int tc_chunks(int W) { return 2 * ((TC_POS + (W - 1) + TC_STAGE - 1) / TC_STAGE); }   /* even: two per stage */
size_t tc_smem_bytes(int W) { return (size_t)tc_chunks(W) * (512 + TC_CHUNK * sizeof(float)); }
int tc_tile() { return TC_POS; }

cudaError_t launch_reweight_tc(const ReweightParams& prm, unsigned grid, cudaStream_t stream)
{
    const size_t smem = tc_smem_bytes(prm.W);
    if (smem > 48 * 1024) {
        const cudaError_t e = cudaFuncSetAttribute(umi_reweight_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    umi_reweight_tc_kernel<<<grid, TC_THREADS, smem, stream>>>(prm, tc_chunks(prm.W));
    return cudaGetLastError();
}

} // namespace umi
