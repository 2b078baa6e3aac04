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

/* ---- programmatic dependent launch (sm_90+): the reweighting kernel is launched with
   cudaLaunchAttributeProgrammaticStreamSerialization, so its CTAs may start -- and stage their samples, which do
   not depend on the median kernel -- while the median kernel's last CTAs are still running; it waits here before
   it touches what the median kernel wrote.  Both instructions do nothing in a launch without the attribute. ---- */
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait_for_primary() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

/* ---- sm_100a packed fp32x2 arithmetic (FFMA2 / FMUL2 / FADD2): two fp32 in one 64-bit register pair ---- */
typedef unsigned long long f32x2;                    /* two fp32 in one 64-bit register pair */

__device__ __forceinline__ f32x2 pack2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 ffma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 fmul2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 fadd2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}


/* -min(|u_eff|, 1) from nu = -u and au = alpha*u (Eq. 2-3).  Exactly one of the two is
   <= 0 and that one is -|u_eff|; compared as signed integers a non-positive float is below every
   positive one and, among non-positive floats, a larger magnitude is a larger integer, so the
   three-input integer minimum with bits(-1.0f) selects -|u_eff| and clamps it at -1 in one DPX
   instruction (VIMNMX3).  NaN inputs come out as -1 (weight 0), like the float form did. */
__device__ __forceinline__ float neg_ueff_clamped(float nu, float au)
{
    return __int_as_float(__vimin3_s32(__float_as_int(nu), __float_as_int(au), (int)0xBF800000));
}

/* The same when alpha = 2^APOW exactly (alpha = 2 is the paper's default): alpha*u = -alpha*nu
   is then ONE integer add on the bit pattern of nu -- 0x80000000 flips the sign, APOW << 23 raises the
   exponent -- so the multiply leaves the FMA pipe, which is the pipe that limits the kernel, for the ALU
   pipe (VIADDMNMX = min(nu + const, nu), then VIMNMX with -1.0f).  Bit-identical to the multiply for
   every normal nu with |nu| < 2^(127-APOW); zero / denormal nu give a |u_eff| below 2^-125 either way
   (weight exactly 1); the callers route windows in which nu could overflow (k * tile range >= 2^100) to
   the multiply form, because a nu of -Inf or NaN would wrap to a small value here instead of to weight 0. */
template <int APOW>
__device__ __forceinline__ float neg_ueff_clamped_pow2(float nu)
{
    constexpr int ADDC = (int)(0x80000000u + ((unsigned)APOW << 23));
    const int i = __float_as_int(nu);
    return __int_as_float(__vimin3_s32(i, i + ADDC, (int)0xBF800000));
}

/* Phase 3 (Eq. 2-4) on two samples of one position at once, on u' = -u: S2 += w, R2 += w*u' per half
   (the caller negates the sum).  kn2 = (-k, -k), cn2 = (-c0, -c0), nalpha2 = (-alpha, -alpha).
   APOW < 0: any alpha; APOW >= 0: alpha = 2^APOW (nalpha2 unused). */
template <int APOW>
__device__ __forceinline__ void eval_weight_pair(f32x2 x2, f32x2 kn2, f32x2 cn2, f32x2 nalpha2,
                                                 f32x2& S2, f32x2& R2)
{
    const f32x2 a2 = ffma2(x2, kn2, cn2);                /* -u */
    float a0, a1;
    unpack2(a2, a0, a1);
    f32x2 ne2;
    if constexpr (APOW >= 0) {
        ne2 = pack2(neg_ueff_clamped_pow2<APOW>(a0), neg_ueff_clamped_pow2<APOW>(a1));
    } else {
        const f32x2 b2 = fmul2(a2, nalpha2);             /* alpha*u */
        float b0, b1;
        unpack2(b2, b0, b1);
        ne2 = pack2(neg_ueff_clamped(a0, b0), neg_ueff_clamped(a1, b1));
    }
    const f32x2 n2 = ffma2(ne2, ne2, pack2(-1.f, -1.f)); /* -(1 - e^2) <= 0: Eq. 3 cut-off already applied (R12) */
    const f32x2 w2 = fmul2(n2, n2);
    S2 = fadd2(S2, w2);
    R2 = ffma2(w2, a2, R2);
}

/* alpha = 2^m for m in {0, 1, 2} -> m, else -1 (which compiled variant of the passes a launch takes) */
__host__ __device__ inline int alpha_pow2(float alpha)
{
    return alpha == 1.f ? 0 : alpha == 2.f ? 1 : alpha == 4.f ? 2 : -1;
}

} // namespace umi

#endif
