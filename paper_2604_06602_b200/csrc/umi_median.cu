/*
 * umi_median.cu -- Phase 1: exact sliding-window sample median.
 *
 * CTA = one star x one tile of T consecutive positions.  The T windows of a tile
 * live inside one union of U = T + W - 1 = NS samples.  The union is sorted ONCE
 * per tile (bitonic, 64-bit key|index), then each lane of one warp walks T/32
 * consecutive positions, keeping the union-rank of the current window's median:
 * a slide removes one sample and adds one, so the median moves by at most a
 * couple of included ranks.  Exact (the result is a selected sample);
 * O(log^2 U) per position for the sort plus O(1) expected per slide, instead of
 * O(W) per position for a per-thread quickselect (the paper's kernel).
 * Readings R1-R6, R16, R18 of DESIGN.md.  Nothing here is shared with oracle/.
 */
#include "umi_device.cuh"

namespace umi {

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

} // namespace umi
