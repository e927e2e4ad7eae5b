// dbie_math.cuh — per-interaction arithmetic of the DBIE kernel (Eq. 6):
//   geometry  r^2 -> 1/r, r, 1/r^3
//   kernel    n(theta) = theta sin(theta) + cos(theta), theta = |lambda| r >= 0   (A3)
//             by a 256-entry table of (sin, cos)(k pi/128) plus short polynomials on |t| <= pi/256
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
// them with UMOV / IMAD.MOV pairs in the inner loop.
#if defined(__CUDACC__)
static __constant__ double kTrigC[11] = {DBIE_SIN_S0, DBIE_SIN_S1, DBIE_COS_C0, DBIE_COS_C1,
                                         DBIE_COS_C2, DBIE_INV_STEP, DBIE_STEP_HI, DBIE_ROUND_MAGIC,
                                         DBIE_SINR_S0, DBIE_COSR_C0, DBIE_COSR_C1};
#endif
#if defined(__CUDA_ARCH__) && !defined(DBIE_COEF_IMMEDIATE)
#define DBIE_K(i, name) ::dbie::kTrigC[i]
#else
#define DBIE_K(i, name) (name)
#endif

// (sin, cos)(k pi/128), k = 0..255, correctly rounded (gen_trig_coeffs.py).  The kernels keep
// kTrigCopies interleaved copies in shared memory (entry k of copy g at index k*8 + g) and lane l
// reads copy l & 7: the 8 lanes of a quarter-warp then hit 8 different 16-byte bank groups whatever
// their k, so the LDS.128 of the lookup never has a bank conflict.  The host build has one copy.
constexpr int kTrigEntries = DBIE_TRIG_ENTRIES;
struct TrigEntry {
    double s, c;
};
constexpr int kTrigCopies = 8;
#if !defined(__CUDA_ARCH__)
static const TrigEntry kTrigTabHost[kTrigEntries] = {DBIE_TRIG_TABLE};
#endif
#if defined(__CUDACC__)
static __device__ const TrigEntry kTrigTabG[kTrigEntries] = {DBIE_TRIG_TABLE};
#endif
constexpr int kTrigTableBytes = kTrigEntries * kTrigCopies * (int)sizeof(TrigEntry);   // 32 KB
struct TrigRef {
    const TrigEntry* e;   // host: the table; device: the CTA's shared-memory table (copy 0)
    unsigned lane_off;    // device: byte offset of this lane's copy, (lane & 7) * 16
};

DBIE_HD int lo32(double v) {
#if defined(__CUDA_ARCH__)
    return __double2loint(v);
#else
    uint64_t b;
    memcpy(&b, &v, 8);
    return (int)(uint32_t)b;
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
// 5 FP64-pipe instructions + 1 MUFU; the last step is y0 * (1 + e p) rather than fma(y0 e, p, y0) so that
// no instruction reads three different registers (one more rounding: <= 1 ulp instead of 0.5).
DBIE_HD double rsqrt_full(double a) {
    const double y0 = rsqrt_seed(a);
    const double ay = a * y0;
    const double e = fma(-ay, y0, 1.0);
    const double p = fma(e, 0.375, 0.5);
    const double g = fma(e, p, 1.0);
    return y0 * g;
}

// sin and cos of the REDUCED argument t, |t| <= pi/256 (1.0005 slack): 7 FP64 instructions.
// Approximation error 2e-19 / 2e-21 absolute (trig_coeffs.h).  sin t = t + t (u S(u)) keeps t in two
// operand slots of the last FMA: every FP64 instruction here reads at most two different registers
// (a DFMA with three different register operands costs three issue cycles instead of two on B200,
// profiles/r02_fp64_operand_probe.md).
// REDUCED (reading A-12, dbie_eval with DBIE_EVAL_REDUCED_SINCOS only; never the solver): one coefficient
// fewer in each polynomial, 5 instructions, approximation error 3.0e-13 (sin) / 1.8e-16 (cos) absolute.
template <bool REDUCED = false>
DBIE_HD void sincos_small(double t, double& sn, double& cs) {
    const double u = t * t;
    if (REDUCED) {
        sn = fma(t, u * DBIE_K(8, DBIE_SINR_S0), t);
        cs = fma(u, fma(DBIE_K(10, DBIE_COSR_C1), u, DBIE_K(9, DBIE_COSR_C0)), 1.0);
        return;
    }
    const double p = fma(DBIE_K(1, DBIE_SIN_S1), u, DBIE_K(0, DBIE_SIN_S0));
    sn = fma(t, u * p, t);
    double q = fma(DBIE_K(4, DBIE_COS_C2), u, DBIE_K(3, DBIE_COS_C1));
    q = fma(q, u, DBIE_K(2, DBIE_COS_C0));
    cs = fma(u, q, 1.0);
}

// Reduction theta = k pi/128 + t for 0 <= theta < 2^20.  One Cody-Waite step with the double
// nearest to pi/128: the FMA forms theta - k*STEP_HI exactly and rounds once.  The neglected tail
// k*(pi/128 - STEP_HI) = theta * 3.9e-17 is the same as evaluating sin/cos at theta (1 + 3.9e-17):
// a perturbation that is smooth in theta (no jump at interval boundaries) and below the
// half-ulp rounding (1.1e-16 theta) that theta = |lambda| r already carries.  3 FP64 instructions;
// k is read from the low word of the magic-number sum, so no FP64<->int conversion.
DBIE_HD double reduce_step(double th, int& k) {
    const double kf = fma(th, DBIE_K(5, DBIE_INV_STEP), DBIE_ROUND_MAGIC);
    k = lo32(kf);
    const double kd = kf - DBIE_ROUND_MAGIC;
    return fma(-kd, DBIE_K(6, DBIE_STEP_HI), th);
}

DBIE_HD TrigEntry trig_entry(const TrigRef& tr, int k) {
#if defined(__CUDA_ARCH__)
    // byte offset ((k & 255) * 128) | lane_off from the CTA-uniform base: IMAD.SHL + one LOP3 + LDS.128 [R + UR]
    const unsigned off = (((unsigned)k << 7) & (unsigned)((kTrigEntries - 1) << 7)) | tr.lane_off;
    const double2 v = *reinterpret_cast<const double2*>(reinterpret_cast<const unsigned char*>(tr.e) + off);
    return TrigEntry{v.x, v.y};
#else
    return tr.e[k & (kTrigEntries - 1)];
#endif
}

// n(theta) = theta sin(theta) + cos(theta), theta >= 0 (Eq. 6 numerator).  16 FP64
// instructions, no quadrant logic.  With (S, C) = (sin, cos)(k pi/128) from the table and (sn, cs) =
// (sin, cos)(t):  sin theta = S cs + C sn, cos theta = C cs - S sn, so
//   n = cs (theta S + C) + sn (theta C - S).
template <bool REDUCED = false>
DBIE_HD double kernel_n(double th, const TrigRef& tr) {
    int k;
    const double t = reduce_step(th, k);
    const TrigEntry e = trig_entry(tr, k);
    double sn, cs;
    sincos_small<REDUCED>(t, sn, cs);
    const double a = fma(th, e.s, e.c);
    const double b = fma(th, e.c, -e.s);
    return fma(cs, a, sn * b);
}

// n(theta) and cos(theta): the analytic-gradient mode (O-5).  18 FP64 instructions.
DBIE_HD void kernel_n_cos(double th, const TrigRef& tr, double& n, double& c) {
    int k;
    const double t = reduce_step(th, k);
    const TrigEntry e = trig_entry(tr, k);
    double sn, cs;
    sincos_small(t, sn, cs);
    const double a = fma(th, e.s, e.c);
    const double b = fma(th, e.c, -e.s);
    n = fma(cs, a, sn * b);
    c = fma(e.c, cs, -(e.s * sn));
}

// (sin, cos)(eps) for |eps| <= 1e-3: sin eps = eps - eps^3/6 (next term eps^5/120 <= 8e-18), cos eps = 1 - eps^2/2 +
// eps^4/24 (next term eps^6/720 <= 1.4e-21).  5 FP64 instructions.
DBIE_HD void sincos_tiny(double eps, double& se, double& ce) {
    const double e2 = eps * eps;
    ce = fma(e2, fma(e2, 1.0 / 24.0, -0.5), 1.0);
    se = fma(eps * e2, -1.0 / 6.0, eps);
}

// n(theta) = theta sin(theta) + cos(theta) at theta = theta0 + eps from (s0, c0) = (sin, cos)(theta0):
//   n = s0 (theta cos eps - sin eps) + c0 (theta sin eps + cos eps).
// 9 FP64 instructions instead of the 16 of a full kernel_n, formed without cancellation against n(theta0); what the
// Eq. 13 stencil uses for the three offset positions of a field point.
DBIE_HD double kernel_n_near(double th, double s0, double c0, double eps) {
    double se, ce;
    sincos_tiny(eps, se, ce);
    const double p = fma(th, ce, -se);
    const double q = fma(th, se, ce);
    return fma(s0, p, c0 * q);
}
constexpr double kNearEpsMax = 1e-3;   // largest |lambda delta| for which the Eq. 13 stencil uses kernel_n_near

// sin(theta) and cos(theta), theta >= 0: 15 FP64 instructions (the Eq. 13 stencil and the GRID trials start from these)
DBIE_HD void sincos_pos(double th, const TrigRef& tr, double& s, double& c) {
    int k;
    const double t = reduce_step(th, k);
    const TrigEntry e = trig_entry(tr, k);
    double sn, cs;
    sincos_small(t, sn, cs);
    s = fma(e.s, cs, e.c * sn);
    c = fma(e.c, cs, -(e.s * sn));
}

}  // namespace dbie
