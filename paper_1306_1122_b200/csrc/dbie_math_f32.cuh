// dbie_math_f32.cuh — fp32 per-interaction arithmetic of dbie_eval_f32 (Eq. 6;
// BASELINE.json config 4 "fp64 and fp32").  Same structure as dbie_math.cuh:
//   geometry  r^2 -> 1/r (MUFU.RSQ, 2^-22), r, 1/r^3
//   kernel    n(theta) = theta sin(theta) + cos(theta), theta = |lambda| r >= 0
// Two ways to get (sin, cos), chosen per component at compile time:
//   SFU : two-term reduction by 2 pi, then MUFU.SIN / MUFU.COS of the REDUCED argument (|t| <= pi,
//         where their absolute error is 2^-21.4), so the error does not grow with theta and no quadrant
//         logic is needed: 10 FP32-pipe instructions + 2 MUFU per component;
//   TAB : the fp64 kernel's scheme in fp32 — theta = k pi/128 + t, (sin, cos)(k pi/128) from the 256-entry table
//         (float copy, 16 interleaved copies in shared memory so that the LDS.64 of a half-warp never conflicts),
//         sin t = t - t^3/6, cos t = 1 - t^2/2 on |t| <= pi/256: 15 FP32-pipe instructions, no MUFU.
// Mixing them balances the SFU (16 lanes/clk/SM) against the issue port.
// __host__ __device__ so the host shim can check TAB against mpmath (the SFU path is device only).
#pragma once
#include <math.h>
#include <stdint.h>
#include <string.h>

#include "trig_coeffs.h"
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

struct TrigEntryF {
    float s, c;
};
constexpr int kTrigCopiesF = 16;
constexpr int kTrigTableBytesF = DBIE_TRIG_ENTRIES * kTrigCopiesF * (int)sizeof(TrigEntryF);   // 32 KB
#if !defined(__CUDA_ARCH__)
static const TrigEntryF kTrigTabHostF[DBIE_TRIG_ENTRIES] = {DBIE_TRIG_TABLE};   // the fp64 table, rounded to float
#endif
#if defined(__CUDACC__)
static __device__ const TrigEntryF kTrigTabGF[DBIE_TRIG_ENTRIES] = {DBIE_TRIG_TABLE};
#endif
struct TrigRefF {
    const TrigEntryF* e;   // host: the table; device: the CTA's shared-memory table (copy 0)
    unsigned lane_off;     // device: byte offset of this lane's copy, (lane & 15) * 8
};

DBIE_HD32 TrigEntryF trig_entry_f32(const TrigRefF& tr, int k) {
#if defined(__CUDA_ARCH__)
    const unsigned off = (((unsigned)k << 7) & (unsigned)((DBIE_TRIG_ENTRIES - 1) << 7)) | tr.lane_off;
    const float2 v = *reinterpret_cast<const float2*>(reinterpret_cast<const unsigned char*>(tr.e) + off);   // LDS.64
    return TrigEntryF{v.x, v.y};
#else
    return tr.e[k & (DBIE_TRIG_ENTRIES - 1)];
#endif
}

template <bool SFU>
DBIE_HD32 float kernel_n_f32(float th, const TrigRefF& tr) {
#if defined(__CUDA_ARCH__)
    if (SFU) {
        // theta = k 2 pi + t, |t| <= pi, where MUFU.SIN / MUFU.COS are good to 2^-21.4 absolute: no quadrant
        // logic at all, n = theta sin t + cos t.
        const float kf = fmaf(th, DBIE_F32_INV_TWOPI, DBIE_F32_ROUND_MAGIC);
        const float kd = kf - DBIE_F32_ROUND_MAGIC;
        float t = fmaf(-kd, DBIE_F32_TWOPI_HI, th);
        t = fmaf(-kd, DBIE_F32_TWOPI_LO, t);
        return fmaf(th, __sinf(t), __cosf(t));
    }
#endif
    // theta = k pi/128 + t: k from the low mantissa bits of the magic-number sum (no F2I), two-term Cody-Waite
    const float kf = fmaf(th, DBIE_F32_INV_STEP, DBIE_F32_ROUND_MAGIC);
    const int k = f32_bits(kf);
    const float kd = kf - DBIE_F32_ROUND_MAGIC;
    float t = fmaf(-kd, DBIE_F32_STEP_HI, th);
    t = fmaf(-kd, DBIE_F32_STEP_LO, t);
    const TrigEntryF e = trig_entry_f32(tr, k);
    const float u = t * t;
    const float sn = fmaf(t * u, -1.0f / 6.0f, t);
    const float cs = fmaf(u, -0.5f, 1.0f);
    const float a = fmaf(th, e.s, e.c);
    const float b = fmaf(th, e.c, -e.s);
    return fmaf(cs, a, sn * b);
}

}  // namespace dbie
