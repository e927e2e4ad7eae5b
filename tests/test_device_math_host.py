"""Host-side checks of the CUDA path's own arithmetic (no GPU, no oracle).

`paper_1306_1122_b200/csrc/dbie_math.cuh` and `dbie_nm.cuh` are __host__ __device__; the host
shim compiles them with g++ so that the polynomial sincos, the reciprocal-sqrt refinement, the
per-interaction term, the residual formulas and the resumable Nelder-Mead state machine can be
checked here against mpmath / NumPy / SciPy.  Nothing under oracle/ is imported.
"""
import ctypes as C
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import optimize

from paper_1306_1122_b200 import build as dbuild

_dp = C.POINTER(C.c_double)


@pytest.fixture(scope="module")
def shim():
    lib = C.CDLL(dbuild.build_hostshim())
    lib.shim_nm_generic.restype = C.c_int
    return lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _ulp(x):
    return np.spacing(np.abs(x))


def test_trig_coefficients_header_is_current():
    import subprocess, sys, os
    script = os.path.join(os.path.dirname(dbuild.__file__), "csrc", "gen_trig_coeffs.py")
    subprocess.check_call([sys.executable, script, "--check"])


def test_sincos_accuracy_against_mpmath(shim):
    """|theta| up to 1000 rad (config 4 reaches ~155): error <= 1.5 ulp of the result + the reduced
    argument's rounding + the one-step Cody-Waite tail theta*(pi/128 - fl(pi/128))/(pi/128) = 3.9e-17 theta,
    which stays below the half-ulp rounding 1.1e-16 theta that theta = |lambda| r itself carries
    (dbie_math.cuh reduce_pio2)."""
    rng = np.random.default_rng(1)
    th = np.concatenate([rng.uniform(0, 2, 2000), rng.uniform(0, 200, 4000), rng.uniform(0, 1000, 2000),
                         np.arange(0, 400) * (math.pi / 4), np.arange(1, 400) * (math.pi / 2) * (1 + 1e-12),
                         [0.0, 1e-300, 1e-8, 0.7853981633974483, 0.7853981633974484]])
    s = np.empty_like(th); c = np.empty_like(th)
    shim.shim_sincos(C.c_long(th.size), _p(th), _p(s), _p(c))
    mp.mp.dps = 50
    worst = 0.0
    for t, si, ci in zip(th, s, c):
        es, ec = mp.sin(mp.mpf(float(t))), mp.cos(mp.mpf(float(t)))
        # error budget: 1.5 ulp of the value + the roundings of the table entries and of the two products that
        # combine them with (sin t, cos t) (1.2e-16 absolute)
        for got, ex in ((si, es), (ci, ec)):
            err = abs(mp.mpf(float(got)) - ex)
            tol = 1.5 * float(_ulp(float(ex))) + 1.2e-16 + 4.0e-17 * float(t)
            worst = max(worst, float(err / tol))
    assert worst <= 1.0, worst


def test_kernel_n_matches_definition(shim):
    """n(theta) = theta sin(theta) + cos(theta): within 3e-16 (|theta|+1) plus the
    one-step Cody-Waite tail, |dn/dtheta| * 3.9e-17 theta <= 4e-17 theta^2 (the rounding of
    theta = |lambda| r contributes 1.1e-16 theta^2 before the kernel ever sees it)."""
    rng = np.random.default_rng(2)
    th = np.concatenate([rng.uniform(0, 160, 5000), [0.0, 1e-9, 0.5, 100.0]])
    out = np.empty_like(th)
    shim.shim_kernel_n(C.c_long(th.size), _p(th), _p(out))
    mp.mp.dps = 50
    for t, got in zip(th, out):
        ex = mp.mpf(float(t)) * mp.sin(mp.mpf(float(t))) + mp.cos(mp.mpf(float(t)))
        assert abs(mp.mpf(float(got)) - ex) <= 3e-16 * (float(t) + 1.0) + 4e-17 * float(t) ** 2
    # evenness is taken care of by the caller (|lambda|); n(0) = 1 exactly
    assert out[-4] == 1.0


def test_kernel_n_reduced_sincos_error(shim):
    """The eval-only reduced-degree variant (reading A-12; DBIE_EVAL_REDUCED_SINCOS): its error on n(theta) is the
    sin polynomial's 3.0e-13 times theta (n = theta sin + cos), far inside what dbie_eval's 1e-9 on B allows."""
    rng = np.random.default_rng(12)
    th = np.concatenate([rng.uniform(0, 400, 6000), [0.0, 1e-9]])
    out = np.empty_like(th)
    full = np.empty_like(th)
    shim.shim_kernel_n_reduced(C.c_long(th.size), _p(th), _p(out))
    shim.shim_kernel_n(C.c_long(th.size), _p(th), _p(full))
    mp.mp.dps = 40
    worst = 0.0
    for t, got in zip(th, out):
        ex = mp.mpf(float(t)) * mp.sin(mp.mpf(float(t))) + mp.cos(mp.mpf(float(t)))
        worst = max(worst, float(abs(mp.mpf(float(got)) - ex)) / (float(t) + 1.0))
    assert 1e-14 < worst <= 3.5e-13, worst          # really the reduced polynomials, and within their bound
    assert out[-2] == 1.0 and np.abs(out - full).max() > 0


def test_kernel_n_cos_matches_definition(shim):
    """kernel_n_cos (analytic-gradient mode, O-5): n(theta) as kernel_n, bit for bit, and cos(theta)."""
    rng = np.random.default_rng(13)
    th = rng.uniform(0, 300, 3000)
    n = np.empty_like(th); c = np.empty_like(th); n0 = np.empty_like(th)
    shim.shim_kernel_n_cos(C.c_long(th.size), _p(th), _p(n), _p(c))
    shim.shim_kernel_n(C.c_long(th.size), _p(th), _p(n0))
    assert np.array_equal(n, n0)
    mp.mp.dps = 40
    for t, got in zip(th, c):
        assert abs(mp.mpf(float(got)) - mp.cos(mp.mpf(float(t)))) <= 3.5e-16 + 4e-17 * float(t)


def test_trig_table_is_correctly_rounded():
    """The 256-entry (sin, cos)(k pi/128) table of trig_coeffs.h: every entry is the double nearest to the exact
    value (exact 0, +-1 at the multiples of pi/2)."""
    import os
    import re
    path = os.path.join(os.path.dirname(dbuild.__file__), "csrc", "trig_coeffs.h")
    text = open(path).read()
    body = text[text.index("#define DBIE_TRIG_TABLE"):]
    pairs = re.findall(r"\{([-+0-9.e]+), ([-+0-9.e]+)\}", body)
    assert len(pairs) == 256
    mp.mp.dps = 50
    for k, (sv, cv) in enumerate(pairs):
        a = 2 * mp.pi * k / 256
        for got, ex in ((float(sv), mp.sin(a)), (float(cv), mp.cos(a))):
            if k % 64 == 0:
                assert got == float(round(ex))
            else:
                assert got == float(ex)             # mpmath -> float conversion rounds to nearest


def test_rsqrt_refinement(shim):
    rng = np.random.default_rng(3)
    a = np.concatenate([10.0 ** rng.uniform(-6, 8, 5000), [1.0, 4.0, 2.0, 1e-30, 1e30]])
    out = np.empty_like(a)
    shim.shim_rsqrt(C.c_long(a.size), _p(a), _p(out))
    mp.mp.dps = 50
    rel = [abs(mp.mpf(float(o)) * mp.sqrt(mp.mpf(float(x))) - 1) for x, o in zip(a, out)]
    # the last step is y0 * (1 + e p) (two roundings: no FP64 instruction with three different register
    # operands), so the bound is 1 ulp + the product's half ulp at worst
    assert max(rel) <= 3.4e-16, float(max(rel))


def test_single_interaction_term(shim):
    """One (point, pixel) term as the kernel's inner loop forms it vs the definition in mpmath."""
    rng = np.random.default_rng(4)
    mp.mp.dps = 40
    for _ in range(300):
        dx, dy = rng.uniform(-400, 400, 2)
        z = rng.uniform(0.5, 200)
        lam = rng.uniform(-0.2, 0.2, 3)
        b0 = rng.uniform(-1500, 1500, 3)
        out = np.empty(3)
        shim.shim_interaction(C.c_double(dx), C.c_double(dy), C.c_double(z), _p(lam), _p(b0), _p(out))
        r = mp.sqrt(mp.mpf(dx) ** 2 + mp.mpf(dy) ** 2 + mp.mpf(z) ** 2)
        for p in range(3):
            th = abs(mp.mpf(lam[p])) * r
            ex = (th * mp.sin(th) + mp.cos(th)) / r ** 3 * mp.mpf(b0[p])
            scale = (float(th) + 1.0) / float(r) ** 3 * abs(b0[p])
            # theta = fl(lambda * r) carries 2^-53 * theta of angle error (same in the oracle)
            assert abs(mp.mpf(out[p]) - ex) <= 4e-16 * scale * max(1.0, float(th)), (dx, dy, z, p)


def test_residual_formulas(shim):
    """Eq. 8, 9, 13, 14 re-derived with NumPy."""
    rng = np.random.default_rng(5)
    for _ in range(50):
        Bs = rng.normal(0, 1, (4, 3))
        Bs[1:] = Bs[0] + 1e-3 * rng.normal(0, 1, (3, 3))
        delta, d, wg = 1e-3, 1.0, 0.7
        out = np.empty(7)
        shim.shim_residual(_p(Bs.ravel().copy()), C.c_double(delta), C.c_double(d), C.c_double(wg), _p(out))
        G = (Bs[1:] - Bs[0]).T / delta            # G[p, j] = dB_p/dx_j
        J = np.array([G[2, 1] - G[1, 2], G[0, 2] - G[2, 0], G[1, 0] - G[0, 1]])
        div = np.trace(G)
        B = Bs[0]
        f = np.linalg.norm(np.cross(J, B)) / (np.linalg.norm(J) * np.linalg.norm(B))
        g = abs(div) * (d / 6) / np.linalg.norm(B)
        assert np.allclose(out[2:5], J, rtol=1e-13, atol=0)
        assert np.isclose(out[5], div, rtol=1e-12, atol=1e-12)
        assert np.isclose(out[0], f, rtol=1e-12) and np.isclose(out[1], g, rtol=1e-12)
        assert np.isclose(out[6], f + wg * g, rtol=1e-12)
    # |B| = 0 is an invalid point
    out = np.empty(7)
    shim.shim_residual(_p(np.zeros(12)), C.c_double(1e-3), C.c_double(1.0), C.c_double(1.0), _p(out))
    assert np.isnan(out[6])


_OBJ = C.CFUNCTYPE(C.c_double, _dp)


def _run_nm(shim, fn, simplex, xtol, ftol, maxiter):
    cb = _OBJ(lambda p: float(fn(np.array([p[0], p[1], p[2]]))))
    simplex = np.ascontiguousarray(simplex, dtype=np.float64)
    trace = np.full((maxiter + 1, 3), np.nan)
    fs = np.empty((4, 3)); ff = np.empty(4)
    it, nf = C.c_int(), C.c_int()
    st = shim.shim_nm_generic(cb, _p(simplex), C.c_double(xtol), C.c_double(ftol), C.c_int(maxiter),
                              _p(trace), _p(fs), _p(ff), C.byref(it), C.byref(nf))
    return {"status": st, "iters": it.value, "nfev": nf.value, "simplex": fs, "f": ff,
            "trace": trace[: it.value + 1]}


@pytest.mark.parametrize("name", ["quadratic", "rosenbrock3", "abs_kink"])
def test_nm_state_machine_matches_scipy(shim, name):
    """The resumable state machine reproduces SciPy's non-adaptive Nelder-Mead vertex for vertex."""
    fns = {
        "quadratic": lambda v: (v[0] - 0.3) ** 2 + 2 * (v[1] + 0.1) ** 2 + 0.5 * (v[2] - 0.7) ** 2
                               + 0.3 * v[0] * v[1],
        "rosenbrock3": lambda v: 100 * (v[1] - v[0] ** 2) ** 2 + (1 - v[0]) ** 2
                                 + 100 * (v[2] - v[1] ** 2) ** 2 + (1 - v[1]) ** 2,
        "abs_kink": lambda v: abs(v[0] - 0.2) + abs(v[1] + 0.4) ** 1.5 + (v[2] - 0.1) ** 2 + 0.05 * math.sin(9 * v[0]),
    }
    fn = fns[name]
    x0 = np.array([0.05, 0.05, 0.05])
    simplex = np.vstack([x0, x0 + [0.05, 0, 0], x0 + [0, 0.05, 0], x0 + [0, 0, 0.05]])
    xtol, ftol, maxiter = 1e-6, 1e-9, 400
    mine = _run_nm(shim, fn, simplex, xtol, ftol, maxiter)
    best = []
    res = optimize.minimize(fn, x0, method="Nelder-Mead",
                            options={"initial_simplex": simplex, "adaptive": False, "xatol": xtol,
                                     "fatol": ftol, "maxiter": maxiter + 1, "maxfev": 10 ** 6,
                                     "return_all": True})
    best = np.array(res.allvecs)
    # SciPy starts its counter at 1 (nit = 1 + simplex updates) and records allvecs[0] before
    # its initial sort
    assert mine["iters"] == res.nit - 1
    assert mine["nfev"] == res.nfev
    assert mine["status"] == (1 if res.status == 0 else 2)
    assert np.array_equal(mine["trace"][1:], best[1: mine["iters"] + 1])
    assert np.array_equal(mine["simplex"], res.final_simplex[0])
    assert np.array_equal(mine["f"], res.final_simplex[1])


def test_nm_maxiter_and_shrink_paths(shim):
    """A function with a narrow curved valley exercises contraction and shrink; maxiter stops it."""
    calls = []

    def fn(v):
        calls.append(tuple(v))
        return (v[0] ** 2 + v[1] ** 2 + v[2] ** 2 - 1) ** 2 + 5 * abs(v[0] - v[1]) + abs(v[2])
    x0 = np.array([1.0, -1.0, 0.5])
    simplex = np.vstack([x0, x0 + [0.3, 0, 0], x0 + [0, 0.3, 0], x0 + [0, 0, 0.3]])
    mine = _run_nm(shim, fn, simplex, 1e-10, 1e-14, 60)
    res = optimize.minimize(fn, x0, method="Nelder-Mead",
                            options={"initial_simplex": simplex, "adaptive": False, "xatol": 1e-10,
                                     "fatol": 1e-14, "maxiter": 61, "maxfev": 10 ** 6})
    assert mine["iters"] == res.nit - 1 == 60 and mine["status"] == 2
    assert mine["nfev"] == res.nfev
    assert np.array_equal(mine["simplex"][0], res.x)


def test_kernel_n_f32_table_path(shim):
    """fp32 n(theta) = theta sin theta + cos theta of dbie_math_f32.cuh (angle-table path, no MUFU) against
    mpmath at the float inputs: |error| <= 4 ulp_f32(theta) + 2e-7 for theta up to 400 rad
    (config 4 reaches ~155).  The dominant term is theta * (error of sin) ~ theta * 6e-8."""
    rng = np.random.default_rng(5)
    th = np.concatenate([rng.uniform(0, 2, 1000), rng.uniform(0, 160, 4000), rng.uniform(0, 400, 1000),
                         np.arange(0, 200) * (math.pi / 4), [0.0, 1e-20, 0.78539816]]).astype(np.float32)
    out = np.empty_like(th)
    fp = C.POINTER(C.c_float)
    shim.shim_kernel_n_f32(C.c_long(th.size), th.ctypes.data_as(fp), out.ctypes.data_as(fp))
    mp.mp.dps = 30
    worst = 0.0
    for t, got in zip(th, out):
        tt = mp.mpf(float(t))
        ex = tt * mp.sin(tt) + mp.cos(tt)
        tol = 4.0 * float(np.spacing(np.float32(max(float(t), 1.0)))) + 2e-7
        worst = max(worst, float(abs(mp.mpf(float(got)) - ex)) / tol)
    assert worst <= 1.0, worst


def test_kernel_n_near_against_mpmath(shim):
    """n(theta0 + eps) from (sin, cos)(theta0), the form the Eq. 13 stencil uses for its three offset positions:
    within a few ulp of theta for exact inputs, and the DIFFERENCE n(theta0 + eps) - n(theta0) - what the finite
    differences divide by delta - to a relative 1e-11 of its own size (no cancellation between the positions)."""
    rng = np.random.default_rng(16)
    n = 3000
    th0 = rng.uniform(0.5, 300, n)
    eps = np.concatenate([rng.uniform(-1e-3, 1e-3, n // 2), rng.uniform(-1e-4, 1e-4, n // 2)])
    mp.mp.dps = 40
    s0 = np.array([float(mp.sin(mp.mpf(t))) for t in th0]); c0 = np.array([float(mp.cos(mp.mpf(t))) for t in th0])
    th = th0 + eps
    out = np.empty(n)
    shim.shim_kernel_n_near(C.c_long(n), _p(th), _p(s0), _p(c0), _p(eps), _p(out))
    for i in range(n):
        e, T = mp.mpf(float(eps[i])), mp.mpf(float(th[i]))
        S0, C0 = mp.mpf(float(s0[i])), mp.mpf(float(c0[i]))
        S, Cc = S0 * mp.cos(e) + C0 * mp.sin(e), C0 * mp.cos(e) - S0 * mp.sin(e)    # exact rotation of the given pair
        ex = T * S + Cc
        assert abs(mp.mpf(float(out[i])) - ex) <= 3e-16 * (float(th[i]) + 1.0)
