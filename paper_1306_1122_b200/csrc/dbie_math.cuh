// dbie_math.cuh — per-interaction arithmetic of the DBIE kernel (Eq. 6):
//   geometry  r^2 -> 1/r, r, 1/r^3
//   kernel    n(theta) = theta sin(theta) + cos(theta), theta = |lambda| r >= 0   (A3)
// Everything is written with explicit fma()/__dmul-style operations so the FP64-pipe
// instruction count is what the source says (DESIGN.md section 6 counts them).
// The functions are __host__ __device__ so that tests/test_device_math_host.py can run the
// very same arithmetic on the CPU against mpmath (only the reciprocal-sqrt seed differs).
#pragma once
#include <math.h>
#include <stdint.h>
#include <string.h>

#include "trig_coeffs.h"

#if defined(__CUDACC__)
#define DBIE_HD __host__ __device__ __forceinline__
#else
#define DBIE_HD inline
#endif

namespace dbie {

DBIE_HD int lo32(double v) {
#if defined(__CUDA_ARCH__)
    return __double2loint(v);
#else
    uint64_t b;
    memcpy(&b, &v, 8);
    return (int)(uint32_t)b;
#endif
}

DBIE_HD double flip_sign_if(double v, int bit31) {  // bit31 is 0 or 0x80000000
#if defined(__CUDA_ARCH__)
    return __hiloint2double(__double2hiint(v) ^ bit31, __double2loint(v));
#else
    uint64_t b;
    memcpy(&b, &v, 8);
    b ^= (uint64_t)(uint32_t)bit31 << 32;
    memcpy(&v, &b, 8);
    return v;
#endif
}

// Seed of 1/sqrt(a), relative error <= 2^-22 (MUFU.RSQ64H on the device).
DBIE_HD double rsqrt_seed(double a) {
#if defined(__CUDA_ARCH__)
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    return y;
#else
    return (double)(float)(1.0 / sqrt(a));  // host stand-in with a comparable error (2^-24)
#endif
}

// 1/sqrt(a) to ~1 ulp for normal a > 0: one third-order step on the seed.
//   e = 1 - a y0^2,  y1 = y0 (1 + e/2 + 3 e^2/8);  seed error eps -> 2.5 eps^3 (< 2^-64).
// 5 FP64-pipe instructions + 1 MUFU.
DBIE_HD double rsqrt_full(double a) {
    const double y0 = rsqrt_seed(a);
    const double ay = a * y0;
    const double e = fma(-ay, y0, 1.0);
    const double p = fma(e, 0.375, 0.5);
    const double q = y0 * e;
    return fma(q, p, y0);
}

// sin and cos of the REDUCED argument t, |t| <= pi/4 (1.0005 slack): 14 FP64 instructions.
DBIE_HD void sincos_reduced(double t, double& sn, double& cs) {
    const double u = t * t;
    double s = DBIE_SIN_S5;
    s = fma(s, u, DBIE_SIN_S4);
    s = fma(s, u, DBIE_SIN_S3);
    s = fma(s, u, DBIE_SIN_S2);
    s = fma(s, u, DBIE_SIN_S1);
    s = fma(s, u, DBIE_SIN_S0);
    double c = DBIE_COS_C5;
    c = fma(c, u, DBIE_COS_C4);
    c = fma(c, u, DBIE_COS_C3);
    c = fma(c, u, DBIE_COS_C2);
    c = fma(c, u, DBIE_COS_C1);
    c = fma(c, u, DBIE_COS_C0);
    const double tu = t * u;
    sn = fma(tu, s, t);
    cs = fma(u, c, 1.0);
}

// Reduction theta = k pi/2 + t for 0 <= theta < 2^20 (two-term Cody-Waite; with an FMA the
// first step is exact while k < 2^20).  4 FP64 instructions; the
// quadrant is read from the low word of the magic-number sum, so no FP64<->int conversion.
DBIE_HD double reduce_pio2(double th, int& q) {
    const double kf = fma(th, DBIE_TWO_OVER_PI, DBIE_ROUND_MAGIC);
    q = lo32(kf);
    const double kd = kf - DBIE_ROUND_MAGIC;
    double t = fma(-kd, DBIE_PIO2_HI, th);
    t = fma(-kd, DBIE_PIO2_LO, t);
    return t;
}

// n(theta) = theta sin(theta) + cos(theta), theta >= 0 (Eq. 6 numerator).
// 19 FP64 instructions.
DBIE_HD double kernel_n(double th) {
    int q;
    const double t = reduce_pio2(th, q);
    double sn, cs;
    sincos_reduced(t, sn, cs);
    // quadrant q&3: sin(theta), cos(theta) = (sn,cs), (cs,-sn), (-sn,-cs), (-cs,sn).
    // Selects and sign flips are integer-pipe work (FSEL/LOP3), not FP64-pipe instructions.
    const bool odd = (q & 1) != 0;
    const double a = odd ? cs : sn;
    const double b = flip_sign_if(odd ? sn : cs, q << 31);
    const double n = fma(th, a, b);
    return flip_sign_if(n, (q << 30) & (int)0x80000000);
}

// full sincos (used by host accuracy tests and by nothing on the hot path)
DBIE_HD void sincos_pos(double th, double& s, double& c) {
    int q;
    const double t = reduce_pio2(th, q);
    double sn, cs;
    sincos_reduced(t, sn, cs);
    const bool odd = (q & 1) != 0;
    const double a = odd ? cs : sn;
    const double b = flip_sign_if(odd ? sn : cs, q << 31);
    const int sg = (q << 30) & (int)0x80000000;
    s = flip_sign_if(a, sg);
    c = flip_sign_if(b, sg);
}

}  // namespace dbie
