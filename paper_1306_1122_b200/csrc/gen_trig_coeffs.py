"""Generate the polynomial coefficients and the angle table of the device sincos (trig_coeffs.h).

The interaction kernel needs sin(theta) and cos(theta) for theta = lambda*r >= 0
(Eq. 6 numerator theta*sin(theta) + cos(theta)).  fp64: after a one-step
Cody-Waite reduction theta = k*(pi/128) + t, |t| <= pi/256, the kernel reads
(sin, cos)(k pi/128) from a 256-entry table (one period) and evaluates

    sin t = t + t*t^2 * S(t^2)          S of degree NS-1 in u = t^2   (NS = 2)
    cos t = 1 + t^2 * C(t^2)            C of degree NC-1 in u = t^2   (NC = 3)

(fp32 variant: the same table rounded to float with two-term polynomials, or MUFU.SIN/COS after a reduction by 2 pi.)  This script computes S and C as
weighted minimax polynomials (Remez exchange, mpmath, 60 digits), rounds them to double, reports
the approximation error of the ROUNDED coefficients, and writes trig_coeffs.h with the correctly
rounded table.  Run:

    python paper_1306_1122_b200/csrc/gen_trig_coeffs.py [--check]

The header is committed; the build does not run this script.
"""
from __future__ import annotations

import os
import struct
import sys

import mpmath as mp

mp.mp.dps = 60
HERE = os.path.dirname(os.path.abspath(__file__))
TAB_N = 256                               # table entries over one period: step 2 pi / 256 = pi / 128
A = (mp.pi / 4) * mp.mpf("1.0005")        # |t| bound with slack for the rounding of k (set per variant below)
UA = A * A


def set_interval(a):
    global A, UA
    A = a
    UA = A * A


def g_sin(u):
    """(sin(t)/t - 1)/u with u = t^2."""
    if u < mp.mpf("1e-20"):
        return -mp.mpf(1) / 6 + u / 120
    t = mp.sqrt(u)
    return (mp.sin(t) / t - 1) / u


def g_cos(u):
    """(cos(t) - 1)/u with u = t^2."""
    if u < mp.mpf("1e-20"):
        return -mp.mpf(1) / 2 + u / 24
    t = mp.sqrt(u)
    return (mp.cos(t) - 1) / u


def horner(c, u):
    r = mp.mpf(0)
    for a in reversed(c):
        r = r * u + a
    return r


def remez(g, n, weight, iters=30):
    """Minimax degree-(n-1) polynomial p(u) on [0, UA] minimising max |weight(u) (p - g)(u)|."""
    # initial reference: Chebyshev extrema mapped to [0, UA] (avoid u = 0 where weight may vanish)
    m = n + 1
    xs = [UA * (1 - mp.cos(mp.pi * (i + mp.mpf("0.5")) / m)) / 2 for i in range(m)]
    coeffs = None
    for _ in range(iters):
        # solve p(x_i) + (-1)^i E / w(x_i) = g(x_i)
        Mx = mp.matrix(m, m)
        rhs = mp.matrix(m, 1)
        for i, x in enumerate(xs):
            for j in range(n):
                Mx[i, j] = x ** j
            Mx[i, n] = (-1) ** i / weight(x)
            rhs[i] = g(x)
        sol = mp.lu_solve(Mx, rhs)
        coeffs = [sol[j] for j in range(n)]
        err = lambda u: weight(u) * (horner(coeffs, u) - g(u))
        # locate the extrema of the error on a fine grid, one per sign run
        K = 4000
        grid = [UA * i / K for i in range(1, K + 1)]
        vals = [err(u) for u in grid]
        runs = []
        cur = [0]
        for i in range(1, K):
            if (vals[i] > 0) == (vals[cur[-1]] > 0):
                cur.append(i)
            else:
                runs.append(cur)
                cur = [i]
        runs.append(cur)
        ext = [max(r, key=lambda i: abs(vals[i])) for r in runs]
        if len(ext) < m:
            break
        # keep the m consecutive extrema with the largest minimum magnitude
        best = max(range(len(ext) - m + 1), key=lambda s: min(abs(vals[i]) for i in ext[s:s + m]))
        new = [grid[i] for i in ext[best:best + m]]
        if max(abs(a - b) for a, b in zip(new, xs)) < UA * mp.mpf("1e-12"):
            xs = new
            break
        xs = new
    return coeffs


def to_double(x):
    return float(x)


def hexbits(d):
    return "0x%016x" % struct.unpack("<Q", struct.pack("<d", d))[0]


def report(name, coeffs_d, exact, approx_from):
    """Max abs error of the rounded-coefficient approximation, in units of 2^-53."""
    K = 3000
    worst = mp.mpf(0)
    for i in range(K + 1):
        t = A * i / K
        e = abs(approx_from(coeffs_d, t) - exact(t))
        worst = max(worst, e)
    return worst


def sin_from(c, t):
    u = t * t
    return t + t * u * horner([mp.mpf(a) for a in c], u)


def cos_from(c, t):
    u = t * t
    return 1 + u * horner([mp.mpf(a) for a in c], u)


def split_hi_lo(x, zero_low_bits=0):
    hi = float(x)
    if zero_low_bits:
        b = struct.unpack("<Q", struct.pack("<d", hi))[0]
        b &= ~((1 << zero_low_bits) - 1)
        hi = struct.unpack("<d", struct.pack("<Q", b))[0]
    lo = float(x - mp.mpf(hi))
    return hi, lo


def to_float(x):
    return struct.unpack("<f", struct.pack("<f", float(x)))[0]


def hexbits32(f):
    return "0x%08x" % struct.unpack("<I", struct.pack("<f", f))[0]


def f32_header():
    """fp32 variant (dbie_eval_f32): reduction constants of its two sincos paths.  The table path uses the fp64
    header's DBIE_TRIG_TABLE rounded to float, with sin t = t - t^3/6, cos t = 1 - t^2/2 on |t| <= pi/256."""
    step = 2 * mp.pi / TAB_N
    shi = to_float(step)
    slo = to_float(step - mp.mpf(shi))
    tp = to_float(2 * mp.pi)
    lines = [
        "// GENERATED by gen_trig_coeffs.py -- do not edit.",
        "#pragma once",
        "#define DBIE_F32_ROUND_MAGIC 12582912.0f  /* 1.5 * 2^23 */",
        "// table path: theta = k (pi/128) + t, |t| <= pi/256; truncation of sin t = t - t^3/6: 2.3e-12, of cos t = 1 - t^2/2: 9.5e-10",
        "#define DBIE_F32_INV_STEP %sf  /* 128/pi  %s */" % (repr(to_float(1 / step)), hexbits32(to_float(1 / step))),
        "#define DBIE_F32_STEP_HI %sf  /* pi/128  %s */" % (repr(shi), hexbits32(shi)),
        "#define DBIE_F32_STEP_LO %sf  /* %s */" % (repr(slo), hexbits32(slo)),
        "// SFU path: theta = k 2 pi + t, |t| <= pi (MUFU.SIN/COS: 2^-21.4 absolute on [-pi, pi])",
        "#define DBIE_F32_INV_TWOPI %sf  /* %s */" % (repr(to_float(1 / (2 * mp.pi))), hexbits32(to_float(1 / (2 * mp.pi)))),
        "#define DBIE_F32_TWOPI_HI %sf  /* %s */" % (repr(tp), hexbits32(tp)),
        "#define DBIE_F32_TWOPI_LO %sf  /* %s */" % (repr(to_float(2 * mp.pi - mp.mpf(tp))),
                                                      hexbits32(to_float(2 * mp.pi - mp.mpf(tp)))),
        "",
    ]
    return "\n".join(lines)


def main():
    set_interval((mp.pi / TAB_N) * mp.mpf("1.0005"))
    out = {}
    for ns in (2, 3):
        c = remez(g_sin, ns, lambda u: u * mp.sqrt(u))      # error enters as t^3 * (S - g)
        cd = [to_double(a) for a in c]
        out[("S", ns)] = (cd, report("sin", cd, mp.sin, sin_from))
    for nc in (2, 3, 4):
        c = remez(g_cos, nc, lambda u: u)                   # error enters as t^2 * (C - g)
        cd = [to_double(a) for a in c]
        out[("C", nc)] = (cd, report("cos", cd, mp.cos, cos_from))
    for k, (cd, e) in out.items():
        print(k, "max abs approx error = %.3e (%.3f x 2^-53)" % (float(e), float(e * 2 ** 53)))
    NS, NC = 2, 3
    S, C = out[("S", NS)][0], out[("C", NC)][0]
    # eval-only reduced variant (reading A-12; DBIE_EVAL_REDUCED_SINCOS): one coefficient fewer in each
    SR = [to_double(a) for a in remez(g_sin, 1, lambda u: u * mp.sqrt(u))]
    ESR = report("sin", SR, mp.sin, sin_from)
    CR, ECR = out[("C", 2)]
    print("reduced: sin %.3e cos %.3e" % (float(ESR), float(ECR)))
    step_hi, step_lo = split_hi_lo(2 * mp.pi / TAB_N)
    inv_step = float(TAB_N / (2 * mp.pi))
    lines = [
        "// GENERATED by gen_trig_coeffs.py (weighted Remez, mpmath 60 digits) -- do not edit.",
        "// theta = k (pi/128) + t: (sin, cos)(k pi/128) from DBIE_TRIG_TABLE (correctly rounded), and",
        "// sin t = t + t*t^2*S(t^2), cos t = 1 + t^2*C(t^2) on |t| <= pi/256 (1.0005 slack).",
        "// approximation error of the rounded coefficients: sin %.2e, cos %.2e (absolute)."
        % (float(out[("S", NS)][1]), float(out[("C", NC)][1])),
        "#pragma once",
        "#define DBIE_TRIG_NS %d" % NS,
        "#define DBIE_TRIG_NC %d" % NC,
        "#define DBIE_TRIG_ENTRIES %d" % TAB_N,
    ]
    for i, a in enumerate(S):
        lines.append("#define DBIE_SIN_S%d %s  /* %s */" % (i, repr(a), hexbits(a)))
    for i, a in enumerate(C):
        lines.append("#define DBIE_COS_C%d %s  /* %s */" % (i, repr(a), hexbits(a)))
    lines.append("// reduced variant: sin t = t + t*t^2*SR0, cos t = 1 + t^2*(CR0 + CR1 t^2); approximation error sin %.2e, cos %.2e"
                 % (float(ESR), float(ECR)))
    lines.append("#define DBIE_SINR_S0 %s  /* %s */" % (repr(SR[0]), hexbits(SR[0])))
    for i, a in enumerate(CR):
        lines.append("#define DBIE_COSR_C%d %s  /* %s */" % (i, repr(a), hexbits(a)))
    lines += [
        "#define DBIE_INV_STEP %s  /* 128/pi  %s */" % (repr(inv_step), hexbits(inv_step)),
        "#define DBIE_STEP_HI %s  /* pi/128  %s */" % (repr(step_hi), hexbits(step_hi)),
        "#define DBIE_STEP_LO %s  /* %s */" % (repr(step_lo), hexbits(step_lo)),
        "#define DBIE_ROUND_MAGIC 6755399441055744.0  /* 1.5 * 2^52 */",
        "// {sin, cos}(k pi/128), k = 0..255, each rounded to nearest",
        "#define DBIE_TRIG_TABLE \\",
    ]
    for k in range(TAB_N):
        a = 2 * mp.pi * k / TAB_N
        sv, cv = float(mp.sin(a)), float(mp.cos(a))
        if k % (TAB_N // 4) == 0:                        # exact values at the multiples of pi/2
            sv, cv = float(round(mp.sin(a))), float(round(mp.cos(a)))
        lines.append("    {%s, %s}%s" % (repr(sv), repr(cv), ", \\" if k + 1 < TAB_N else ""))
    lines.append("")
    text = "\n".join(lines)
    for name, body in (("trig_coeffs.h", text), ("trig_coeffs_f32.h", f32_header())):
        path = os.path.join(HERE, name)
        if "--check" in sys.argv:
            with open(path) as fh:
                assert fh.read() == body, name + " is stale"
            print(name, "up to date")
        else:
            with open(path, "w") as fh:
                fh.write(body)
            print("wrote", path)


if __name__ == "__main__":
    main()
