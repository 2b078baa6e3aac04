/*
 * umi_median.cu -- Phase 1: exact sliding-window sample median.
 *
 * CTA = one star x one tile of T consecutive positions.  The T windows of a tile
 * live inside one union of U = T + W - 1 = NS samples (NS a power of two).
 *   1. sort the 32-bit keys of the union ONCE per tile: bitonic network, E = NS/THREADS keys per
 *      thread (128 threads of 8 at NS = 1024, 256 threads beyond) -- strides < E in registers, strides < 32 E with warp shuffles, only the top three
 *      strides through shared memory; a compare-exchange is two VIMNMX.  What is sorted is
 *      (key - smallest key of the tile) << log2 NS | union index whenever that fits 32 bits (the
 *      keys of a tile normally span 2^17 .. 2^21 values): rank and index of every entry are then
 *      read off the sorted words.  Otherwise (a wild sample, a deep eclipse in the tile) the bare
 *      keys are sorted and the rank of an entry is the lower bound of its key in the sorted keys
 *      (binary search in shared memory) plus its turn among the entries with the same key (a
 *      shared-memory counter per key value).  Either way srt[rank] = key << 32 | index and
 *      rank[index] come out.  (Sorting 64-bit key|index entries directly cost 4-6 instructions
 *      per exchange and two shuffles.)
 *   2. NW "walkers" (one thread each) own T/NW consecutive positions.  A walker's
 *      first window is selected from a bitset of the union ranks it holds; the NW
 *      bitsets are built together as an exclusive-or prefix scan over the entries
 *      that leave / enter between consecutive walkers (2 T atomicXor per tile
 *      instead of NW W), and the median is the k-th set bit (popcount + fns);
 *   3. each walker then slides: one sample leaves, one enters, so the union rank of
 *      the median moves by at most a couple of included ranks (O(1) expected).
 * Exact: the result is a selected input sample.  O(log^2 U) per position for the
 * sort instead of O(W) per position for a per-thread quickselect (the paper's
 * kernel).  Readings R1-R6, R16, R18 of DESIGN.md.
 * Nothing here is shared with oracle/.
 */
#include "umi_device.cuh"

/* UMI_K1_RADIX = 1 (python -m paper_2604_06602_b200.build --define UMI_K1_RADIX=1) replaces the bitonic network + rank search by
   least-significant-digit radix passes; measured and not the default: 0.82 against 0.63 ms on config 2, 9.13 against 7.25 ms on
   20,000 config-5 stars */
#ifndef UMI_K1_RADIX
#define UMI_K1_RADIX 0
#endif
#ifndef UMI_K1_BITWALK
#define UMI_K1_BITWALK 1
#endif
#ifndef UMI_K1_TRANSPOSED_SCATTER
#define UMI_K1_TRANSPOSED_SCATTER 1
#endif

namespace umi {

namespace {


/* 32-bit keys: one compare-exchange is two VIMNMX (the direction is a predicate operand), one exchange
   with another lane is one shuffle and one VIMNMX.  Equal keys are harmless here: min / max keep the
   multiset, and the ranks of tied entries are assigned after the sort (see the kernel). */
__device__ __forceinline__ void cmp_swap(uint32_t& a, uint32_t& b, bool up)
{
    const uint32_t lo = up ? min(a, b) : max(a, b);                 /* one VIMNMX each: the direction is its predicate operand */
    const uint32_t hi = up ? max(a, b) : min(a, b);
    a = lo;
    b = hi;
}

/* index of sorted key i in skey[]: one pad word per 32 keys, so that the probes of the rank search -- all at
   i = -1 (mod 32) in its first steps -- fall into different banks (they were 75 % of the kernel's bank conflicts) */
__device__ __forceinline__ int skey_at(int i) { return i + (i >> 5); }

/* E consecutive slots of one star row starting at cadence j (j = 0 mod 4 when vec): keys, KEY_INVALID where invalid */
template <int E>
__device__ __forceinline__ int load_keys(const double* __restrict__ trow, const float* __restrict__ frow, int64_t N, int64_t j,
                                         bool vec, uint32_t (&key)[E])
{
    int nvalid = 0;
    if (E % 4 == 0 && vec) {
#pragma unroll
        for (int e = 0; e + 3 < E; e += 4) {
            const int64_t jj = j + e;
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            bool in = jj >= 0 && jj < N;                            /* a group of 4 lies entirely inside or outside the row */
            bool t0 = in, t1 = in, t2 = in, t3 = in;
            if (in) {
                v = __ldg(reinterpret_cast<const float4*>(frow + jj));
                if (trow != nullptr) {
                    const double2 ta = __ldg(reinterpret_cast<const double2*>(trow + jj));
                    const double2 tb = __ldg(reinterpret_cast<const double2*>(trow + jj + 2));
                    t0 = finite_f64(ta.x); t1 = finite_f64(ta.y); t2 = finite_f64(tb.x); t3 = finite_f64(tb.y);
                }
            }
            t0 = t0 && finite_f32(v.x); t1 = t1 && finite_f32(v.y); t2 = t2 && finite_f32(v.z); t3 = t3 && finite_f32(v.w);
            key[e] = t0 ? float_to_key(v.x) : KEY_INVALID;
            key[e + 1] = t1 ? float_to_key(v.y) : KEY_INVALID;
            key[e + 2] = t2 ? float_to_key(v.z) : KEY_INVALID;
            key[e + 3] = t3 ? float_to_key(v.w) : KEY_INVALID;
            nvalid += (int)t0 + (int)t1 + (int)t2 + (int)t3;
        }
    } else {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            float x = 0.f;
            const bool ok = load_sample(trow, frow, N, j + e, x);
            nvalid += ok ? 1 : 0;
            key[e] = ok ? float_to_key(x) : KEY_INVALID;
        }
    }
    return nvalid;
}

/* One bitonic stage (merge size K, stride J) on keys i = tid*E + e held in v[e] (blocked). */
template <int E, int K, int J>
__device__ __forceinline__ void bitonic_stage(uint32_t (&v)[E], uint32_t* buf, int tid)
{
    if constexpr (J < E) {
        /* partner inside the thread */
#pragma unroll
        for (int e = 0; e < E; ++e) {
            if ((e & J) == 0) {
                const bool up = (K < E) ? ((e & K) == 0) : (((tid * E) & K) == 0);
                cmp_swap(v[e], v[e | J], up);
            }
        }
    } else if constexpr (J < 32 * E) {
        /* partner in another lane of the warp */
        constexpr int LM = J / E;
        const bool up = ((tid * E) & K) == 0;
        const bool low = (tid & LM) == 0;
        const bool keep_min = (low == up);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const uint32_t o = __shfl_xor_sync(0xFFFFFFFFu, v[e], LM);
            v[e] = keep_min ? min(v[e], o) : max(v[e], o);
        }
    } else {
        /* partner in another warp: exchange through shared memory */
        __syncthreads();
        const bool up = ((tid * E) & K) == 0;
        const bool low = ((tid * E) & J) == 0;
        const bool keep_min = (low == up);
        const uint32_t* other = buf + ((tid * E) ^ J);
        if constexpr (E % 4 == 0) {
            /* 16-byte chunks, chunk c stored at c ^ ((c >> 3) & 7) within its group of 8: with E > 4 a thread's chunks
               are E/4 apart, which would put a quarter-warp's 128-bit accesses on 2 (E = 16) or 4 (E = 8) bank groups */
            auto chunk = [](int c) { return (c & ~7) | ((c ^ (c >> 3)) & 7); };
            uint4* buf4 = reinterpret_cast<uint4*>(buf);
#pragma unroll
            for (int e = 0; e < E; e += 4)
                buf4[chunk((tid * E + e) >> 2)] = make_uint4(v[e], v[e + 1], v[e + 2], v[e + 3]);
            __syncthreads();
#pragma unroll
            for (int e = 0; e < E; e += 4) {
                const uint4 o4 = buf4[chunk((((tid * E) ^ J) + e) >> 2)];
                v[e] = keep_min ? min(v[e], o4.x) : max(v[e], o4.x);
                v[e + 1] = keep_min ? min(v[e + 1], o4.y) : max(v[e + 1], o4.y);
                v[e + 2] = keep_min ? min(v[e + 2], o4.z) : max(v[e + 2], o4.z);
                v[e + 3] = keep_min ? min(v[e + 3], o4.w) : max(v[e + 3], o4.w);
            }
        } else {                                                    /* E = 2 (NS = 512, small batches) */
            *reinterpret_cast<uint2*>(buf + tid * E) = make_uint2(v[0], v[1]);
            __syncthreads();
            const uint2 o2 = *reinterpret_cast<const uint2*>(other);
            v[0] = keep_min ? min(v[0], o2.x) : max(v[0], o2.x);
            v[1] = keep_min ? min(v[1], o2.y) : max(v[1], o2.y);
        }
    }
}

template <int E, int K, int J>
__device__ __forceinline__ void bitonic_merge(uint32_t (&v)[E], uint32_t* buf, int tid)
{
    if constexpr (J > 0) {
        bitonic_stage<E, K, J>(v, buf, tid);
        bitonic_merge<E, K, J / 2>(v, buf, tid);
    }
}

/* Bitonic sort of NS = THREADS*E keys, ascending. */
template <int E, int THREADS, int K = 2>
__device__ __forceinline__ void bitonic_sort_blocked(uint32_t (&v)[E], uint32_t* buf, int tid)
{
    if constexpr (K <= THREADS * E) {
        bitonic_merge<E, K, K / 2>(v, buf, tid);
        bitonic_sort_blocked<E, THREADS, K * 2>(v, buf, tid);
    }
}

} // namespace

/*
 * MAD variant (R21): each walker also keeps the
 * rank range [L, R] of the cnt = (n-1)/2 + 1 window members with the smallest |x - median|; the
 * MAD is the larger of the two end deviations.  The range is contiguous in sorted order and
 * contains the median, so a slide changes it by O(1) members: the leaving / entering sample,
 * then grow / shrink / exchange steps at the two ends.
 */
struct MadRange {
    int L, R, cnt;
};

/* CTAs per SM the registers must allow, per sort length: what the shared memory of that length admits (k1_smem_bytes) */
__host__ __device__ constexpr int k1_min_ctas(int ns) { return ns <= 512 ? 6 : ns == 1024 ? 8 : ns == 2048 ? 4 : ns == 4096 ? 2 : 1; }

template <int E, int THREADS, bool MAD>
__global__ void __launch_bounds__(THREADS, k1_min_ctas(THREADS * E))
umi_median_kernel(MedianParams prm)
{
    constexpr int NS = THREADS * E;
    constexpr bool BITWALK = MAD || UMI_K1_BITWALK;                 /* walkers keep their rank bitsets current through the walk */
    constexpr int BW = NS / 32;                                     /* bitset words per walker */
    constexpr int BWP = BW + 1;                                     /* padded row stride: conflict-free both ways */
    /* walkers per tile (umi_internal.h) */
    constexpr int NW = k1_walkers(NS, MAD);
    constexpr int NWB = NW / 32;                                    /* walker blocks of 32 */
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t* srt = reinterpret_cast<uint64_t*>(smem_raw);          /* [NS] key<<32 | union index, sorted */
    uint16_t* rank = reinterpret_cast<uint16_t*>(srt + NS);         /* [NS] union index -> rank           */
    uint32_t* bits = reinterpret_cast<uint32_t*>(rank + NS);        /* [NW][BWP] rank bitsets, then ...   */
    uint32_t* boff = bits + NW * BWP;                               /* [NWB][BW] block offsets of the scan */
    uint32_t* skey = reinterpret_cast<uint32_t*>(smem_raw + k1_smem_base(NS, MAD, prm.T)) - (NS + NS / 32);   /* [NS + NS/32] sorted keys, padded (skey_at) */
    /* [T] medians of the tile: aliased onto the bitsets, which are dead by then -- except in the MAD build, whose walkers keep
       their bitsets up to date through the walk (below) and stage the medians in the sorted-key area instead (free after the ranks) */
    float* medbuf = BITWALK ? reinterpret_cast<float*>(skey) : reinterpret_cast<float*>(bits);
    /* ... [T] median ranks and [T] window counts behind them (a launch stages either medians or these: in the sorted-key area,
       which holds 4 T bytes but not 8 T, they take the medians' place) */
    uint16_t* rhobuf = BITWALK ? reinterpret_cast<uint16_t*>(medbuf) : reinterpret_cast<uint16_t*>(medbuf + prm.T);
    uint16_t* cntbuf = rhobuf + prm.T;
    float* sclbuf = reinterpret_cast<float*>(smem_raw + k1_smem_base(NS, MAD, prm.T));   /* MAD only: [T] scales */
    __shared__ int s_nvu;
    __shared__ uint32_t s_kmin, s_kmax;                             /* radix path: range of the tile's valid keys */
#if UMI_K1_RADIX
    __shared__ int s_wsum[THREADS / 32];                         /* radix path: warp totals of the digit scan */
#endif

    const int W = prm.W;
    const int T = prm.T;
    const int h = (W - 1) >> 1;
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const bool rows_vec = (prm.N & 3) == 0 && (reinterpret_cast<uintptr_t>(prm.flux) & 15) == 0 &&
                          (reinterpret_cast<uintptr_t>(prm.time) & 15) == 0;

    pdl_launch_dependents();        /* the reweighting kernel may be scheduled once every CTA of this grid has started */

    for (int64_t bid = blockIdx.x; bid < prm.n_blocks; bid += gridDim.x) {
        const int64_t star = bid / prm.tiles_per_star;
        const int64_t tile = bid - star * prm.tiles_per_star;
        const int64_t j0 = tile * T;                                /* first position of the tile */
        const int64_t jbase = j0 - h;                               /* cadence of union index 0 */
        const int64_t rem = prm.N - j0;
        const int Tact = rem < T ? (int)rem : T;
        const float* frow = prm.flux + star * prm.N;
        const double* trow = prm.time ? prm.time + star * prm.N : nullptr;

        if (tid == 0) { s_nvu = 0; s_kmin = 0xFFFFFFFFu; s_kmax = 0u; }
        static_assert((NW * BWP + NWB * BW) % 4 == 0, "the bitset area is zeroed 16 bytes at a time");
        for (int i = tid; i < (NW * BWP + NWB * BW) / 4; i += THREADS) reinterpret_cast<uint4*>(bits)[i] = make_uint4(0u, 0u, 0u, 0u);
        __syncthreads();

        /* 1. load E consecutive union entries and sort their 32-bit keys */
        uint32_t v[E];
        const bool vec = rows_vec && ((jbase + (int64_t)tid * E) & 3) == 0;
        int nvalid = load_keys<E>(trow, frow, prm.N, jbase + (int64_t)tid * E, vec, v);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nvalid += __shfl_xor_sync(0xFFFFFFFFu, nvalid, o);
        if (lane == 0 && nvalid) atomicAdd(&s_nvu, nvalid);
#if UMI_K1_RADIX
        /* Sort by LEAST-SIGNIFICANT-DIGIT RADIX passes on (key - smallest key of the tile): a tile's keys span a narrow
           range (17-21 bits for flux of 1 +- a few per cent), so 2 or 3 passes of at most 9 bits do, where the bitonic
           network needs 55 compare-exchange stages whatever the data.  The entries travel as key << 32 | union index, so
           the last scatter writes srt[] and rank[] directly: no rank search, no tie counters.  One pass:
             rank inside the warp   per round e, lanes with the same digit find each other with match.any; the lowest
                                    of them bumps the warp's own histogram and hands the old count to the others
             scan                   exclusive prefix over (digit, warp), digit-major: thread d owns digit d
             scatter + reload       stable: warp w re-reads positions [32 E w, 32 E (w+1)), element (e, lane) at 32 e + lane
           Invalid entries take no part: the first scatter compacts the valid ones to positions [0, nvu). */
        {
            const int warp = tid >> 5;
            const unsigned lt = (1u << lane) - 1u;
            uint32_t kmn = 0xFFFFFFFFu, kmx = 0u;
            uint64_t el[E];
            bool ok[E];
#pragma unroll
            for (int e = 0; e < E; ++e) {
                ok[e] = v[e] != KEY_INVALID;
                el[e] = ((uint64_t)v[e] << 32) | (uint32_t)(tid * E + e);
                if (ok[e]) { kmn = min(kmn, v[e]); kmx = max(kmx, v[e]); }
                else rank[tid * E + e] = (uint16_t)0xFFFFu;
            }
            kmn = __reduce_min_sync(0xFFFFFFFFu, kmn);
            kmx = __reduce_max_sync(0xFFFFFFFFu, kmx);
            if (lane == 0 && kmn <= kmx) { atomicMin(&s_kmin, kmn); atomicMax(&s_kmax, kmx); }
            __syncthreads();
            const int nv = s_nvu;
            const uint32_t kmin = s_kmin;
            const int nbits = nv > 0 ? 32 - __clz((int)(s_kmax - kmin) | 1) : 1;
            const int passes = (nbits + 8) / 9;
            const int db = (nbits + passes - 1) / passes;           /* digit bits, <= 9 */
            const int nb = 1 << db;
            uint32_t* hist = bits;                                   /* [8 warps][nb] counters, in the bitset area */
            uint32_t* hw = hist + warp * nb;
            for (int pass = 0; pass < passes; ++pass) {
                const int shift = pass * db;
                for (int i = lane; i < nb; i += 32) hw[i] = 0u;
                __syncwarp();
                int off[E];
                uint32_t dig[E];
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const uint32_t d = ok[e] ? ((((uint32_t)(el[e] >> 32) - kmin) >> shift) & (uint32_t)(nb - 1)) : (uint32_t)nb;
                    const unsigned peers = __match_any_sync(0xFFFFFFFFu, d);
                    const int leader = __ffs((int)peers) - 1;
                    uint32_t base = 0u;
                    if (ok[e] && lane == leader) { base = hw[d]; hw[d] = base + (uint32_t)__popc(peers); }
                    base = __shfl_sync(0xFFFFFFFFu, base, leader);
                    off[e] = (int)base + __popc(peers & lt);
                    dig[e] = d;
                    __syncwarp();
                }
                __syncthreads();
                /* exclusive prefix over (digit, warp): thread t owns the digits [t dpt, (t+1) dpt) */
                {
                    const int dpt = nb > THREADS ? nb / THREADS : 1;
                    int mine = 0;
                    for (int j = 0; j < dpt; ++j) {
                        const int d = tid * dpt + j;
                        if (d < nb)
                            for (int w = 0; w < THREADS / 32; ++w) mine += (int)hist[w * nb + d];
                    }
                    int incl = mine;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int t = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                        if (lane >= o) incl += t;
                    }
                    if (lane == 31) s_wsum[warp] = incl;
                    __syncthreads();
                    int run = incl - mine;
                    for (int w = 0; w < warp; ++w) run += s_wsum[w];
                    for (int j = 0; j < dpt; ++j) {
                        const int d = tid * dpt + j;
                        if (d < nb)
                            for (int w = 0; w < THREADS / 32; ++w) {
                                const int c = (int)hist[w * nb + d];
                                hist[w * nb + d] = (uint32_t)run;
                                run += c;
                            }
                    }
                }
                __syncthreads();
                const bool last = pass == passes - 1;
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    if (ok[e]) {
                        const int pos = (int)hw[dig[e]] + off[e];
                        srt[pos] = el[e];
                        if (last) rank[(uint32_t)el[e]] = (uint16_t)pos;
                    }
                }
                __syncthreads();
                if (!last) {
#pragma unroll
                    for (int e = 0; e < E; ++e) {
                        const int pp = warp * (32 * E) + 32 * e + lane;
                        ok[e] = pp < nv;
                        el[e] = ok[e] ? srt[pp] : 0ull;
                    }
                }
            }
            for (int i = tid; i < NW * BWP + NWB * BW; i += THREADS) bits[i] = 0u;   /* the histograms lived in the bitset area */
            __syncthreads();
        }
#else
        constexpr int OWN_MAX = 4;                                  /* (E = 8 spilled with them under its 48-register bound: it reloads, like E = 16 and 32) */
        uint32_t own[E <= OWN_MAX ? E : 1];                               /* the entries' own keys, kept across the sort when they fit */
        if constexpr (E <= OWN_MAX) {
#pragma unroll
            for (int e = 0; e < E; ++e) own[e] = v[e];
        }
        /* The keys of a tile normally span a narrow range (flux of 1 +- a few per cent: 2^17 .. 2^21 key values), so
           (key - smallest key) and the entry's union index fit ONE 32-bit word: sorting those words sorts the entries,
           and each thread reads rank and index of the entries it ends up holding straight off them -- no rank search,
           no tie counters.  Ties come out in index order.  A tile whose keys span 2^(32 - log2 NS) - 1 values or more (a wild
           sample, a deep eclipse) sorts the bare keys and searches, as before. */
        constexpr int LOG_NS = 31 - __builtin_clz((unsigned)NS);
        constexpr uint32_t KSPAN = (1u << (32 - LOG_NS)) - 1u;      /* also: the packed key of an invalid entry */
        {
            uint32_t kmn = 0xFFFFFFFFu, kmx = 0u;
#pragma unroll
            for (int e = 0; e < E; ++e) {
                kmn = min(kmn, v[e]);                               /* KEY_INVALID is the largest word */
                kmx = max(kmx, v[e] != KEY_INVALID ? v[e] : 0u);
            }
            kmn = __reduce_min_sync(0xFFFFFFFFu, kmn);
            kmx = __reduce_max_sync(0xFFFFFFFFu, kmx);
            if (lane == 0 && nvalid) { atomicMin(&s_kmin, kmn); atomicMax(&s_kmax, kmx); }
        }
        __syncthreads();
        const uint32_t kmin = s_kmin;
        const bool pk = s_nvu > 0 && (s_kmax - kmin) < KSPAN;
        if (pk) {
#pragma unroll
            for (int e = 0; e < E; ++e)
                v[e] = ((v[e] != KEY_INVALID ? v[e] - kmin : KSPAN) << LOG_NS) | (uint32_t)(tid * E + e);
        }
        bitonic_sort_blocked<E, THREADS>(v, reinterpret_cast<uint32_t*>(srt), tid);

        if (pk) {
            __syncthreads();                                        /* every read of the exchange buffer (srt) is done */
            /* A thread holds E consecutive ranks: written from there, the 8-byte entries of a warp's lanes lie 8 E bytes apart
               (16-way bank conflicts at E = 8: a fifth of the kernel's shared-memory wavefronts).  So the sorted words take
               one more trip through the exchange buffer (128-bit stores, chunks XOR-swizzled as in the sort) and come back
               striped -- word j THREADS + tid to thread tid -- and consecutive lanes write consecutive entries
               (config 2: 0.557 -> 0.537 ms, config 5: 6.27 -> 6.03 ms per 20,000 stars).  Not at E = 2 (2-way, two barriers more). */
            constexpr bool STRIPED = UMI_K1_TRANSPOSED_SCATTER && (E % 4 == 0);
            if constexpr (STRIPED) {
                uint32_t* wbuf = reinterpret_cast<uint32_t*>(srt);
                auto chunk = [](int c) { return (c & ~7) | ((c ^ (c >> 3)) & 7); };
#pragma unroll
                for (int e = 0; e < E; e += 4)
                    reinterpret_cast<uint4*>(wbuf)[chunk((tid * E + e) >> 2)] = make_uint4(v[e], v[e + 1], v[e + 2], v[e + 3]);
                __syncthreads();
#pragma unroll
                for (int j = 0; j < E; ++j) {
                    const int i = j * THREADS + tid;
                    v[j] = wbuf[4 * chunk(i >> 2) + (i & 3)];
                }
                __syncthreads();                                    /* the words are in registers: srt may be overwritten */
            }
#pragma unroll
            for (int j = 0; j < E; ++j) {
                const int r = STRIPED ? j * THREADS + tid : tid * E + j;
                const uint32_t u = v[j] & (uint32_t)(NS - 1), d = v[j] >> LOG_NS;
                if (d != KSPAN) {
                    rank[u] = (uint16_t)r;
                    srt[r] = ((uint64_t)(kmin + d) << 32) | u;
                } else {
                    rank[u] = (uint16_t)0xFFFFu;
                }
            }
            __syncthreads();
        } else {
#pragma unroll
        for (int e = 0; e < E; ++e) skey[skey_at(tid * E + e)] = v[e];
        __syncthreads();                                            /* also: every read of the exchange buffer is done */

        /* rank of every entry = lower bound of its key among the sorted keys + its turn among the entries
           with that key (a counter per key value, borrowed from the still all-zero bitset area and zeroed
           again below).  Tied entries carry the same value, so which of them gets which rank changes
           nothing that is computed from ranks.  Invalid entries get a rank above every valid one. */
        if constexpr (E > OWN_MAX) (void)load_keys<E>(trow, frow, prm.N, jbase + (int64_t)tid * E, vec, v);   /* the same words again (L1 / L2) */
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int u = tid * E + e;
            const uint32_t key = (E <= OWN_MAX) ? own[(E <= OWN_MAX) ? e : 0] : v[e];
            if (key != KEY_INVALID) {
                int pos = 0;
#pragma unroll
                for (int step = NS / 2; step > 0; step >>= 1)
                    pos += (skey[skey_at(pos + step - 1)] < key) ? step : 0;
                const int r = pos + (int)atomicAdd(&bits[pos], 1u);
                v[e] = (uint32_t)pos;
                rank[u] = (uint16_t)r;
                srt[r] = ((uint64_t)key << 32) | (uint32_t)u;
            } else {
                v[e] = 0xFFFFFFFFu;
                rank[u] = (uint16_t)0xFFFFu;
            }
        }
        __syncthreads();
#pragma unroll
        for (int e = 0; e < E; ++e)
            if (v[e] != 0xFFFFFFFFu) bits[v[e]] = 0u;                  /* the bitset area is all zero again */
        __syncthreads();
        }
#endif
        const int nvu = s_nvu;                                      /* valid entries = ranks [0, nvu) */

        /* 2. walker w owns positions [w*Ts, (w+1)*Ts).  Bitset of the ranks in its first window:
              row 0 = window of position 0; row w = (entries leaving) xor (entries entering) between the
              starts of walkers w-1 and w; an exclusive-or prefix scan over w turns rows into bitsets. */
        const int Ts = (Tact + NW - 1) / NW;
        const int nwa = (Tact + Ts - 1) / Ts;                       /* active walkers */
        const int span = (nwa - 1) * Ts;                            /* start of the last active walker */
        const uint32_t ts_magic = 0xFFFFFFFFu / (uint32_t)Ts + 1u;   /* ceil(2^32 / Ts): u / Ts = umulhi(u, magic), exact while u Ts < 2^32 (Ts = 1: magic wraps to 0, handled) */
        auto walker_of = [&](int u) { return Ts > 1 ? (int)__umulhi((uint32_t)u, ts_magic) : u; };
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int u = tid * E + e;
            const int r = rank[u];
            if (r < nvu) {
                const uint32_t bit = 1u << (r & 31);
                const int wi = r >> 5;
                if (u < W) atomicXor(&bits[wi], bit);
                if (u < span) {
                    const int w = walker_of(u);
                    atomicXor(&bits[(w + 1) * BWP + wi], bit);
                }
                const int ue = u - W;
                if (ue >= 0 && ue < span) {
                    const int w = walker_of(ue);
                    atomicXor(&bits[(w + 1) * BWP + wi], bit);
                }
            }
        }
        __syncthreads();
        /* scan over walkers, one (block of 32 walkers, word column) pair per work item */
        for (int item = tid; item < NWB * BW; item += THREADS) {
            const int col = item % BW, blk = item / BW;
            uint32_t acc = 0u;
            uint32_t* pcol = bits + (blk * 32) * BWP + col;
#pragma unroll 8
            for (int i = 0; i < 32; ++i) {
                acc ^= pcol[i * BWP];
                pcol[i * BWP] = acc;
            }
            boff[item] = acc;                                       /* block total, made exclusive below */
        }
        __syncthreads();
        if (NWB > 1) {
            for (int col = tid; col < BW; col += THREADS) {
                uint32_t acc = 0u;
                for (int blk = 0; blk < NWB; ++blk) {
                    const uint32_t t = boff[blk * BW + col];
                    boff[blk * BW + col] = acc;
                    acc ^= t;
                }
            }
        } else {
            for (int col = tid; col < BW; col += THREADS) boff[col] = 0u;
        }
        __syncthreads();

        /* first window of each walker: n = population of its bitset, median = k-th set bit */
        int n = 0, rho = -1;
        MadRange mr = {0, 0, 0};
        if (tid < nwa) {
            uint32_t* row = bits + tid * BWP;
            const uint32_t* off = boff + (tid >> 5) * BW;
            if constexpr (BITWALK) {                                /* the bitset proper, in place: the walk keeps it current */
#pragma unroll 4
                for (int i = 0; i < BW; ++i) { const uint32_t w0 = row[i] ^ off[i]; row[i] = w0; n += __popc(w0); }
            } else {
#pragma unroll 4
                for (int i = 0; i < BW; ++i) n += __popc(row[i] ^ off[i]);
            }
            auto wd = [&](int i) { return BITWALK ? row[i] : (row[i] ^ off[i]); };      /* word i of my bitset */
            if (n > 0) {
                int need = (n - 1) >> 1;                            /* (R6) lower median */
                for (int i = 0; i < BW; ++i) {
                    const uint32_t word = wd(i);
                    const int pc = __popc(word);
                    if (need < pc) {
                        rho = i * 32 + (int)__fns(word, 0, need + 1);
                        break;
                    }
                    need -= pc;
                }
                if constexpr (MAD) {
                    /* A first guess of the MAD range from the bitset, a whole 32-rank word at a time (about
                       W/U * 32 members each) instead of one member at a time: grow on the side whose word
                       boundary is nearer to the median in value until at least (n-1)/2 + 1 members are inside;
                       mad_fix() below then trims and balances it exactly.  ~NS/64 steps instead of ~W/2. */
                    const int target = ((n - 1) >> 1) + 1;
                    const float med = key_to_float((uint32_t)(srt[rho] >> 32));
                    int wl = rho >> 5, wr = wl;
                    int cnt = __popc(wd(wl));
                    const int wmax = (nvu - 1) >> 5;
                    while (cnt < target) {
                        const bool can_l = wl > 0, can_r = wr < wmax;
                        if (!can_l && !can_r) break;
                        bool left = can_l;
                        if (can_l && can_r) {
                            const float dl = med - key_to_float((uint32_t)(srt[32 * wl - 1] >> 32));
                            const float dr = key_to_float((uint32_t)(srt[32 * (wr + 1)] >> 32)) - med;
                            left = dl <= dr;
                        }
                        if (left) { --wl; cnt += __popc(wd(wl)); }
                        else      { ++wr; cnt += __popc(wd(wr)); }
                    }
                    while ((wd(wl)) == 0u) ++wl;             /* rho's word is inside: both loops stop */
                    while ((wd(wr)) == 0u) --wr;
                    mr.L = 32 * wl + __ffs((int)(wd(wl))) - 1;
                    mr.R = 32 * wr + 31 - __clz((int)(wd(wr)));
                    mr.cnt = cnt;
                }
            }
        }
        __syncthreads();                                            /* bitsets are dead: medbuf reuses them (MAD build: they live on, medbuf is elsewhere) */

        /* 3. walk: a slide removes one entry and adds one */
        if (tid < nwa) {
            const int pbeg = tid * Ts;
            int pend = pbeg + Ts;
            if (pend > Tact) pend = Tact;
            const uint32_t uW = (uint32_t)W;
            int p = pbeg;
            float mad = 0.f;
            /* window members next to rank r, under the window of position q */
            auto val = [&](int r) { return key_to_float((uint32_t)(srt[r] >> 32)); };
            /* MAD build: every slide repairs both ends of the range, several neighbour searches each, so the walker keeps its
               rank bitset current (one bit cleared, one set per slide) and finds the next member with a mask and a count of
               leading / trailing zeros instead of stepping over the ~U/W non-members in between one entry at a time */
            uint32_t* mrow = bits + tid * BWP;
            auto nextm = [&](int r, int q) {
                if constexpr (BITWALK) {
                    int w = (r + 1) >> 5;
                    if (w >= BW) return nvu;
                    uint32_t m = mrow[w] & (0xFFFFFFFFu << ((r + 1) & 31));
                    while (m == 0u) {
                        if (++w >= BW) return nvu;
                        m = mrow[w];
                    }
                    return (w << 5) + __ffs((int)m) - 1;
                } else {
                    do { ++r; } while (r < nvu && ((uint32_t)srt[r] - (uint32_t)q) >= uW);
                    return r;
                }
            };
            auto prevm = [&](int r, int q) {
                if constexpr (BITWALK) {
                    if (r <= 0) return -1;
                    int w = (r - 1) >> 5;
                    uint32_t m = mrow[w] & (0xFFFFFFFFu >> (31 - ((r - 1) & 31)));
                    while (m == 0u) {
                        if (--w < 0) return -1;
                        m = mrow[w];
                    }
                    return (w << 5) + 31 - __clz((int)m);
                } else {
                    do { --r; } while (r >= 0 && ((uint32_t)srt[r] - (uint32_t)q) >= uW);
                    return r;
                }
            };
            /* restore the invariant for window q (median rank rho, n members) and return the MAD */
            auto mad_fix = [&](int q) {
                if (n == 0) { mr.cnt = 0; return 0.f; }
                const int target = ((n - 1) >> 1) + 1;              /* (R21) rank (n-1)/2 of the deviations */
                if (mr.cnt == 0 || rho < mr.L || rho > mr.R) { mr.L = mr.R = rho; mr.cnt = 1; }
                const float med = val(rho);
                const float inf = INFINITY;
                float dL = med - val(mr.L), dR = val(mr.R) - med;
                int Lp = prevm(mr.L, q), Rn = nextm(mr.R, q);
                float dLp = Lp >= 0 ? med - val(Lp) : inf, dRn = Rn < nvu ? val(Rn) - med : inf;
                while (mr.cnt < target) {                           /* grow towards the nearer neighbour */
                    if (dLp <= dRn) { mr.L = Lp; dL = dLp; Lp = prevm(mr.L, q); dLp = Lp >= 0 ? med - val(Lp) : inf; }
                    else            { mr.R = Rn; dR = dRn; Rn = nextm(mr.R, q); dRn = Rn < nvu ? val(Rn) - med : inf; }
                    ++mr.cnt;
                }
                while (mr.cnt > target) {                           /* drop the farther end */
                    if (dL > dR || (dL == dR && mr.L != rho)) { Lp = mr.L; dLp = dL; mr.L = nextm(mr.L, q); dL = med - val(mr.L); }
                    else                                      { Rn = mr.R; dRn = dR; mr.R = prevm(mr.R, q); dR = val(mr.R) - med; }
                    --mr.cnt;
                }
                for (;;) {                                          /* exchange while an outside member is nearer */
                    if (dL > dRn) {
                        Lp = mr.L; dLp = dL; mr.L = nextm(mr.L, q); dL = med - val(mr.L);
                        mr.R = Rn; dR = dRn; Rn = nextm(mr.R, q); dRn = Rn < nvu ? val(Rn) - med : inf;
                    } else if (dR > dLp) {
                        Rn = mr.R; dRn = dR; mr.R = prevm(mr.R, q); dR = val(mr.R) - med;
                        mr.L = Lp; dL = dLp; Lp = prevm(mr.L, q); dLp = Lp >= 0 ? med - val(Lp) : inf;
                    } else {
                        break;
                    }
                }
                return fmaxf(dL, dR);
            };
            if constexpr (MAD) mad = mad_fix(p);
            for (;;) {
                /* emit position p (R4, R5) */
                const bool own = rank[p + h] < nvu;
                const bool has = own && n >= prm.min_valid && n > 0;
                if (!MAD && prm.packed) {                           /* hand-over word, assembled after the walk (never asked of the MAD build) */
                    rhobuf[p] = has ? (uint16_t)rho : (uint16_t)0xFFFFu;
                    cntbuf[p] = (uint16_t)n;
                } else {
                    float m = __int_as_float(0x7FC00000);
                    if (has) m = key_to_float((uint32_t)(srt[rho] >> 32));
                    medbuf[p] = m;
                }
                if constexpr (MAD) sclbuf[p] = has ? mad : __int_as_float(0x7FC00000);
                if (++p >= pend) break;
                /* slide to window p: union index p-1 leaves, p+W-1 enters */
                const int ro = rank[p - 1], ri = rank[p + W - 1];
                const bool vo = ro < nvu, vi = ri < nvu;
                const int n2 = n - (vo ? 1 : 0) + (vi ? 1 : 0);
                if constexpr (BITWALK) {                            /* my bitset becomes that of window p */
                    if (vo) mrow[ro >> 5] &= ~(1u << (ro & 31));
                    if (vi) mrow[ri >> 5] |= 1u << (ri & 31);
                }
                if (n2 == 0) {
                    rho = -1;
                } else if (n == 0) {
                    rho = ri;
                } else {
                    const int k2 = (n2 - 1) >> 1;
                    int below = ((n - 1) >> 1) - ((vo && ro < rho) ? 1 : 0) + ((vi && ri < rho) ? 1 : 0);
                    const uint32_t up = (uint32_t)p;
                    if constexpr (BITWALK) {                        /* the same moves on the bitset */
                        if (vo && ro == rho) {
                            const int r = nextm(rho, p);
                            if (r < nvu) {
                                rho = r;
                            } else {
                                rho = max(prevm(rho, p), 0);
                                --below;
                            }
                        }
                        while (below > k2) { rho = max(prevm(rho, p), 0); --below; }
                        while (below < k2) { rho = min(nextm(rho, p), nvu - 1); ++below; }
                    } else {
                    if (vo && ro == rho) {                          /* the median itself left */
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
                }
                n = n2;
                if constexpr (MAD) {
                    /* the leaving / entering sample against the old range, then repair */
                    /* (the entering one first: moving an end below may land on it) */
                    if (mr.cnt > 0 && vi && ri > mr.L && ri < mr.R) ++mr.cnt;
                    if (mr.cnt > 0 && vo && ro >= mr.L && ro <= mr.R) {
                        if (--mr.cnt > 0) {
                            if (ro == mr.L) mr.L = nextm(mr.L, p);
                            if (ro == mr.R) mr.R = prevm(mr.R, p);
                        }
                    }
                    mad = mad_fix(p);
                }
            }
        }
        __syncthreads();

        float* orow = prm.out + star * prm.N + j0;
        if (!MAD && prm.packed) {
            /* Hand-over word for the reweighting kernel (umi_internal.h), all threads, off the walkers' serial
               chain: where in its window the median sample sits (union index - position, 0 .. W-1), and n+ of
               Eq. 1 (R7) = the n - 1 - (n-1)/2 members above the median in rank, less those that tie with it
               in value (they follow it directly in sorted order). */
            uint32_t* wrow = reinterpret_cast<uint32_t*>(orow);
            for (int p = tid; p < Tact; p += THREADS) {
                const int rho = rhobuf[p];
                uint32_t word = HANDOVER_NONE;
                if (rho != 0xFFFF) {
                    const int n = cntbuf[p];
                    const uint64_t ent = srt[rho];
                    const uint32_t kmed = (uint32_t)(ent >> 32);
                    int np = n - 1 - ((n - 1) >> 1);
                    for (int r = rho + 1; r < nvu && (uint32_t)(srt[r] >> 32) == kmed; ++r)
                        np -= (((uint32_t)srt[r] - (uint32_t)p) < (uint32_t)W) ? 1 : 0;
                    word = ((uint32_t)ent - (uint32_t)p) | ((uint32_t)np << 16);
                }
                wrow[p] = word;
            }
        } else {
            for (int p = tid; p < Tact; p += THREADS) orow[p] = medbuf[p];
        }
        if constexpr (MAD) {
            float* srow = prm.scale + star * prm.N + j0;
            for (int p = tid; p < Tact; p += THREADS) srow[p] = sclbuf[p];
        }
        if (prm.flat != nullptr) {                                  /* PAPER.md:155 normalisation, n_iter = 0 */
            float* flrow = prm.flat + star * prm.N + j0;
            for (int p = tid; p < Tact; p += THREADS) {
                const float m = medbuf[p];
                flrow[p] = (m == m) ? __ldg(frow + j0 + p) / m : m;
            }
        }
        __syncthreads();
    }
}

cudaError_t launch_median(const MedianParams& prm, unsigned grid, size_t smem, cudaStream_t stream)
{
    void (*k1)(MedianParams) = nullptr;
    const bool mad = prm.scale != nullptr;
    int threads = K1_THREADS;
    switch (prm.NS) {
    /* NS = 1024 runs 128 threads of 8 keys: three of the four warps hold walkers (with 256 threads half of the CTA's warps idle
       through the walk), 8 CTAs per SM instead of 6, three of the sort's exchanges in registers instead of two
       (config 2: 0.584 -> 0.558 ms, config 5: 6.78 -> 6.27 ms per 20,000 stars); the longer sorts lose that way */
    case 512: k1 = mad ? umi_median_kernel<2, 256, true> : umi_median_kernel<2, 256, false>; break;
    case 1024: k1 = mad ? umi_median_kernel<8, 128, true> : umi_median_kernel<8, 128, false>; threads = 128; break;
    case 2048: k1 = mad ? umi_median_kernel<8, 256, true> : umi_median_kernel<8, 256, false>; break;
    case 4096: k1 = mad ? umi_median_kernel<16, 256, true> : umi_median_kernel<16, 256, false>; break;
    case 8192: k1 = mad ? umi_median_kernel<32, 256, true> : umi_median_kernel<32, 256, false>; break;
    default: return cudaErrorInvalidValue;
    }
    if (smem + 1024 > 48 * 1024) {        /* static shared memory counts towards the 48 KiB default limit too */
        const cudaError_t e = cudaFuncSetAttribute(k1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    k1<<<grid, threads, smem, stream>>>(prm);
    return cudaGetLastError();
}

} // namespace umi
