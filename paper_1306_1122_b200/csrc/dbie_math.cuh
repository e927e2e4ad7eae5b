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

// On the device the polynomial / reduction constants are read as constant-bank operands of the
// FP64 instructions (DFMA R, R, R, c[3][..]): as 64-bit literals the compiler re-materialises
// them with ~47 UMOV / IMAD.MOV per inner-loop trip (profiles/r01_ncu_full_interact_stencil_cfg2.md).
#if defined(__CUDACC__)
static __constant__ double kTrigC[16] = {
    DBIE_SIN_S0, DBIE_SIN_S1, DBIE_SIN_S2, DBIE_SIN_S3, DBIE_SIN_S4, DBIE_SIN_S5,
    DBIE_COS_C0, DBIE_COS_C1, DBIE_COS_C2, DBIE_COS_C3, DBIE_COS_C4, DBIE_COS_C5,
    DBIE_TWO_OVER_PI, DBIE_PIO2_HI, DBIE_PIO2_LO, DBIE_ROUND_MAGIC};
#endif
#if defined(__CUDA_ARCH__) && !defined(DBIE_COEF_IMMEDIATE)
#define DBIE_K(i, name) ::dbie::kTrigC[i]
#else
#define DBIE_K(i, name) (name)
#endif

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
    double s = DBIE_K(5, DBIE_SIN_S5);
    s = fma(s, u, DBIE_K(4, DBIE_SIN_S4));
    s = fma(s, u, DBIE_K(3, DBIE_SIN_S3));
    s = fma(s, u, DBIE_K(2, DBIE_SIN_S2));
    s = fma(s, u, DBIE_K(1, DBIE_SIN_S1));
    s = fma(s, u, DBIE_K(0, DBIE_SIN_S0));
    double c = DBIE_K(11, DBIE_COS_C5);
    c = fma(c, u, DBIE_K(10, DBIE_COS_C4));
    c = fma(c, u, DBIE_K(9, DBIE_COS_C3));
    c = fma(c, u, DBIE_K(8, DBIE_COS_C2));
    c = fma(c, u, DBIE_K(7, DBIE_COS_C1));
    c = fma(c, u, DBIE_K(6, DBIE_COS_C0));
    const double tu = t * u;
    sn = fma(tu, s, t);
    cs = fma(u, c, 1.0);
}

// Reduction theta = k pi/2 + t for 0 <= theta < 2^20.  One Cody-Waite step with the double
// nearest to pi/2: the FMA forms theta - k*PIO2_HI exactly and rounds once.  The neglected tail
// k*(pi/2 - PIO2_HI) = theta * 3.9e-17 is the same as evaluating sin/cos at theta (1 + 3.9e-17):
// a perturbation that is smooth in theta (no jump at quadrant boundaries) and below the
// half-ulp rounding (1.1e-16 theta) that theta = |lambda| r already carries.  3 FP64 instructions;
// the quadrant is read from the low word of the magic-number sum, so no FP64<->int conversion.
DBIE_HD double reduce_pio2(double th, int& q) {
    const double kf = fma(th, DBIE_K(12, DBIE_TWO_OVER_PI), DBIE_ROUND_MAGIC);
    q = lo32(kf);
    const double kd = kf - DBIE_ROUND_MAGIC;
    return fma(-kd, DBIE_K(13, DBIE_PIO2_HI), th);
}

// n(theta) = theta sin(theta) + cos(theta), theta >= 0 (Eq. 6 numerator).
// 19 FP64 instructions.  Quadrant q&3: (sin, cos)(theta) = (sn,cs), (cs,-sn), (-sn,-cs), (-cs,sn),
// so n = +-(theta sn + cs) for even q and +-(theta cs - sn) for odd q.  Both forms are evaluated
// and one is selected: measured on B200, the extra DFMA is cheaper than swapping the two 64-bit
// operands first (2 FSEL + 1 LOP3 fewer per component; the non-FP64 instructions compete with the
// FP64 pipe for issue slots, profiles/r01_variants.md).
DBIE_HD double kernel_n(double th) {
    int q;
    const double t = reduce_pio2(th, q);
    double sn, cs;
    sincos_reduced(t, sn, cs);
    const double ne = fma(th, sn, cs);
    const double no = fma(th, cs, -sn);
    const double n = (q & 1) ? no : ne;
    return flip_sign_if(n, (q << 30) & (int)0x80000000);
}

// n(theta) and cos(theta) up to their common sign (-1)^(q>>1), which the caller folds into the
// weight: n' in {theta sn + cs, theta cs - sn}, c' in {cs, -sn}; sg = the sign as a bit-31 mask.
// Used by the analytic-gradient mode (O-5).  19 FP64 instructions.
DBIE_HD void kernel_n_cos(double th, double& n, double& c, int& sg) {
    int q;
    const double t = reduce_pio2(th, q);
    double sn, cs;
    sincos_reduced(t, sn, cs);
    const double ne = fma(th, sn, cs);
    const double no = fma(th, cs, -sn);
    const bool odd = (q & 1) != 0;
    n = odd ? no : ne;
    c = odd ? flip_sign_if(sn, (int)0x80000000) : cs;
    sg = (q << 30) & (int)0x80000000;
}

// (sin, cos)(theta0 + eps) from (s0, c0) = (sin, cos)(theta0) for |eps| <= 4e-3: the angle-addition
// formulas with sin eps = eps - eps^3/6 + eps^5/120 (next term 3e-21) and cos eps = 1 - eps^2/2 + eps^4/24
// (next term eps^6/720 <= 6e-18).  11 FP64 instructions instead of the 17 of a full sincos; the
// DIFFERENCE to (s0, c0), which is what Eq. 13's finite differences see, is formed without cancellation.
DBIE_HD void rotate_small(double s0, double c0, double eps, double& s, double& c) {
    const double e2 = eps * eps;
    const double ce = fma(e2, fma(e2, 1.0 / 24.0, -0.5), 1.0);
    const double se = fma(eps * e2, fma(e2, 1.0 / 120.0, -1.0 / 6.0), eps);
    s = fma(s0, ce, c0 * se);
    c = fma(c0, ce, -(s0 * se));
}
constexpr double kRotateSmallMax = 4e-3;

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
