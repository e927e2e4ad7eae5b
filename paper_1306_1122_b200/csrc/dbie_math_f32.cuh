// dbie_math_f32.cuh — fp32 per-interaction arithmetic of dbie_eval_f32 (Eq. 6;
// BASELINE.json config 4 "fp64 and fp32").  Same structure as dbie_math.cuh:
//   geometry  r^2 -> 1/r (MUFU.RSQ, 2^-22), r, 1/r^3
//   kernel    n(theta) = theta sin(theta) + cos(theta), theta = |lambda| r >= 0
// Two ways to get (sin, cos), chosen per component at compile time:
//   POLY: two-term Cody-Waite reduction by pi/2 (exact first step while k < 2^7 ... see below)
//         + minimax polynomials on the FMA pipe (trig_coeffs_f32.h);
//   SFU : two-term reduction by 2 pi, then MUFU.SIN / MUFU.COS of the REDUCED argument (|t| <= pi,
//         where their absolute error is 2^-21.4), so the error does not grow with theta and no quadrant
//         logic is needed.
// __host__ __device__ so the host shim can check POLY against mpmath (the SFU path is device only).
#pragma once
#include <math.h>
#include <stdint.h>
#include <string.h>

#include "trig_coeffs_f32.h"

#if defined(__CUDACC__)
#define DBIE_HD32 __host__ __device__ __forceinline__
#else
#define DBIE_HD32 inline
#endif

namespace dbie {

DBIE_HD32 int f32_bits(float v) {
#if defined(__CUDA_ARCH__)
    return __float_as_int(v);
#else
    int b;
    memcpy(&b, &v, 4);
    return b;
#endif
}
DBIE_HD32 float f32_from_bits(int b) {
#if defined(__CUDA_ARCH__)
    return __int_as_float(b);
#else
    float v;
    memcpy(&v, &b, 4);
    return v;
#endif
}

DBIE_HD32 float rsqrt_f32(float a) {
#if defined(__CUDA_ARCH__)
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(a));
    return y;
#else
    return (float)(1.0 / sqrt((double)a));
#endif
}

// theta = k pi/2 + t.  k = rint(theta 2/pi) through the magic-number sum (its low mantissa
// bits are k, no F2I).  fma(-k, PIO2_HI, theta) is exact: both are multiples of 2^-23 and the
// difference is below 1 (theta < 2^16 keeps k's product within the FMA's exact range).
DBIE_HD32 float reduce_pio2_f32(float th, int& q) {
    const float kf = fmaf(th, DBIE_F32_TWO_OVER_PI, DBIE_F32_ROUND_MAGIC);
    q = f32_bits(kf);
    const float kd = kf - DBIE_F32_ROUND_MAGIC;
    float t = fmaf(-kd, DBIE_F32_PIO2_HI, th);
    t = fmaf(-kd, DBIE_F32_PIO2_LO, t);
    return t;
}

DBIE_HD32 void sincos_reduced_f32(float t, float& sn, float& cs) {
    const float u = t * t;
    float s = DBIE_F32_SIN_S2;
    s = fmaf(s, u, DBIE_F32_SIN_S1);
    s = fmaf(s, u, DBIE_F32_SIN_S0);
    float c = DBIE_F32_COS_C3;
    c = fmaf(c, u, DBIE_F32_COS_C2);
    c = fmaf(c, u, DBIE_F32_COS_C1);
    c = fmaf(c, u, DBIE_F32_COS_C0);
    sn = fmaf(t * u, s, t);
    cs = fmaf(u, c, 1.0f);
}

template <bool SFU>
DBIE_HD32 float kernel_n_f32(float th) {
#if defined(__CUDA_ARCH__)
    if (SFU) {
        // theta = k 2 pi + t, |t| <= pi, where MUFU.SIN / MUFU.COS are good to 2^-21.4 absolute: no quadrant
        // logic at all, n = theta sin t + cos t.  7 FP32-pipe instructions + 2 MUFU per component.
        const float kf = fmaf(th, DBIE_F32_INV_TWOPI, DBIE_F32_ROUND_MAGIC);
        const float kd = kf - DBIE_F32_ROUND_MAGIC;
        float t = fmaf(-kd, DBIE_F32_TWOPI_HI, th);
        t = fmaf(-kd, DBIE_F32_TWOPI_LO, t);
        return fmaf(th, __sinf(t), __cosf(t));
    }
#endif
    int q;
    const float t = reduce_pio2_f32(th, q);
    float sn, cs;
    sincos_reduced_f32(t, sn, cs);
    // both quadrant forms, one selected (as in the fp64 kernel_n): the kernel is issue-bound, and this
    // trades one FSEL + two LOP3/SHF per component for one FFMA
    const float ne = fmaf(th, sn, cs);
    const float no = fmaf(th, cs, -sn);
    const float n = (q & 1) ? no : ne;
    return f32_from_bits(f32_bits(n) ^ ((q << 30) & (int)0x80000000));
}

}  // namespace dbie
