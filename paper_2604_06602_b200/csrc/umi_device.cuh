/* umi_device.cuh -- device helpers shared by the two kernels (validity, key mapping). */
#ifndef UMI_DEVICE_CUH
#define UMI_DEVICE_CUH

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "umi_internal.h"

namespace umi {

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

} // namespace umi

#endif
