"""Pins for the CPU oracle (oracle/dbie_oracle.c) against what the paper and the
mathematics fix — closed forms, invariants, library routines, brute force.
None of these tests touches the CUDA path.  Pin names follow DESIGN.md section 3.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate, optimize

import oracle
from workloads import Workload, config1, dipole_field, random_boundary

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _wl(nx, ny, h, x0, y0, bx, by, bz, pts, lam=None):
    pts = np.atleast_2d(np.asarray(pts, dtype=np.float64))
    M = pts.shape[0]
    lam = np.zeros((3, M)) if lam is None else np.asarray(lam, dtype=np.float64).reshape(3, M)
    return Workload("t", nx, ny, h, x0, y0, np.asarray(bx, float).ravel(),
                    np.asarray(by, float).ravel(), np.asarray(bz, float).ravel(),
                    pts[:, 0].copy(), pts[:, 1].copy(), pts[:, 2].copy(), lam)


def _read_table(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                rows.append([float(t) for t in line.split()])
    return np.array(rows)


# -- K-1 ---------------------------------------------------------------------
def test_k1_one_pixel_worked_example():
    tab = _read_table("k1_one_pixel.txt")
    for lam, want in tab:
        w = _wl(1, 1, 1.0, -0.5, -0.5, [1.0], [1.0], [1.0], [[0.0, 0.0, 1.0]],
                [[lam], [lam], [lam]])
        B = oracle.eval(w)
        assert np.allclose(B[:, 0], want, rtol=0, atol=1e-15)
    # a wrong sign of the sin term, a dropped cos term or 4 pi instead of 2 pi fail here:
    assert abs(tab[2, 1] - (math.sin(1.0) + math.cos(1.0)) / (2 * math.pi)) < 1e-15


# -- K-2 ---------------------------------------------------------------------
def test_k2_kernel_is_normal_derivative_of_reference_function():
    """Eq. 6's kernel equals dY/dz at z=0 of Eq. 5, and the oracle's single-pixel
    term equals h^2 times it (off-axis pixel, all three lambdas different)."""
    mp.mp.dps = 90
    rng = np.random.default_rng(7)
    for _ in range(5):
        xi_f, yi_f = rng.uniform(-3, 3, 2)
        zi_f = rng.uniform(0.5, 4.0)
        xs_f, ys_f = rng.uniform(-3, 3, 2)
        lams = rng.uniform(0.05, 1.5, 3)
        h = 0.25
        xi, yi, zi, xs, ys = (mp.mpf(float(v)) for v in (xi_f, yi_f, zi_f, xs_f, ys_f))
        want = []
        for lam in lams:
            lam = mp.mpf(float(lam))
            def Y(z, lam=lam):
                rho = mp.sqrt((xs - xi) ** 2 + (ys - yi) ** 2 + (z - zi) ** 2)
                rhop = mp.sqrt((xs - xi) ** 2 + (ys - yi) ** 2 + (z + zi) ** 2)
                return mp.cos(lam * rho) / (4 * mp.pi * rho) - mp.cos(lam * rhop) / (4 * mp.pi * rhop)
            dY = mp.diff(Y, 0)
            r = mp.sqrt((xs - xi) ** 2 + (ys - yi) ** 2 + zi ** 2)
            k6 = zi * (lam * r * mp.sin(lam * r) + mp.cos(lam * r)) / (2 * mp.pi * r ** 3)
            assert abs(dY - k6) < mp.mpf(10) ** -30 * abs(k6)
            want.append(float(dY) * h * h)
        b0 = np.array([1.7, -0.4, 2.2])
        w = _wl(1, 1, h, xs_f - h / 2, ys_f - h / 2, [b0[0]], [b0[1]], [b0[2]],
                [[xi_f, yi_f, zi_f]], lams.reshape(3, 1))
        B = oracle.eval(w)[:, 0]
        assert np.allclose(B, np.array(want) * b0, rtol=1e-13, atol=0)


# -- K-3 ---------------------------------------------------------------------
@pytest.mark.parametrize("lam", [0.0, 0.2, 1.0])
def test_k3_radial_gaussian_vs_1d_quadrature(lam):
    """Radially symmetric boundary under the point: the 2-D nodal sum equals
    int_0^inf z n(lam r) r^-3 B0(s) s ds (the 2 pi cancels).  Pins normalisation,
    r, and the whole kernel for lambda != 0 independently of any PDE argument."""
    n, h, sig = 128, 1.0, 5.0
    c = (np.arange(n) + 0.5) * h
    Yg, Xg = np.meshgrid(c, c, indexing="ij")
    xc = yc = 0.5 * n * h
    b0 = np.exp(-((Xg - xc) ** 2 + (Yg - yc) ** 2) / (2 * sig * sig))
    z = 5.0
    w = _wl(n, n, h, 0.0, 0.0, b0, b0, b0, [[xc, yc, z]], [[lam]] * 3)
    got = oracle.eval(w)[0, 0]

    def integrand(s):
        r = math.sqrt(s * s + z * z)
        th = lam * r
        return z * (th * math.sin(th) + math.cos(th)) / r ** 3 * math.exp(-s * s / (2 * sig * sig)) * s
    want, _ = integrate.quad(integrand, 0.0, 60.0, epsabs=0.0, epsrel=1e-12, limit=400)
    assert abs(got - want) <= 1e-10 * abs(want)


# -- K-4 ---------------------------------------------------------------------
def test_k4_uniform_disc_closed_form():
    """B0 = 1 on a disc of radius S under the point:
    integral = cos(lam z) - z cos(lam sqrt(z^2+S^2)) / sqrt(z^2+S^2)
    because d/dr[-cos(lam r)/r] = n(lam r)/r^2.  Pixelised disc converges to it."""
    lam, z = 0.03, 20.0
    errs = []
    for S in (50.0, 200.0):
        n = int(2 * S) + 8
        c = np.arange(n) + 0.5
        Yg, Xg = np.meshgrid(c, c, indexing="ij")
        xc = 0.5 * n
        disc = (((Xg - xc) ** 2 + (Yg - xc) ** 2) <= S * S).astype(float)
        w = _wl(n, n, 1.0, 0.0, 0.0, disc, disc, disc, [[xc, xc, z]], [[lam]] * 3)
        got = oracle.eval(w)[2, 0]
        R = math.sqrt(z * z + S * S)
        want = math.cos(lam * z) - z * math.cos(lam * R) / R
        errs.append(abs(got - want))
    assert errs[1] <= 1e-3
    # independent check of the antiderivative itself by adaptive quadrature
    S = 50.0
    q, _ = integrate.quad(lambda s: z * ((lam * math.hypot(s, z)) * math.sin(lam * math.hypot(s, z))
                                         + math.cos(lam * math.hypot(s, z))) / math.hypot(s, z) ** 3 * s,
                          0.0, S, epsabs=0.0, epsrel=1e-12)
    R = math.hypot(z, S)
    assert abs(q - (math.cos(lam * z) - z * math.cos(lam * R) / R)) < 1e-13


# -- K-5 ---------------------------------------------------------------------
def test_k5_lambda0_rectangle_solid_angle():
    """lambda = 0: Poisson kernel z/(2 pi r^3); uniform rectangle -> Omega / 2 pi.
    Midpoint-rule error at z = 2h is the aliasing term ~ 4 e^{-2 pi z/h} (reading A-2)."""
    n, z = 1001, 2.0
    ones = np.ones(n * n)
    xc = 0.5 * n
    w = _wl(n, n, 1.0, 0.0, 0.0, ones, ones, ones, [[xc, xc, z]])
    got = oracle.eval(w)[2, 0]
    a = b = 0.5 * n
    omega = 4.0 * math.atan(a * b / (z * math.sqrt(a * a + b * b + z * z)))
    want = omega / (2 * math.pi)
    rel = abs(got - want) / want
    predicted = 4.0 * math.exp(-2 * math.pi * z)       # 1.40e-5
    assert abs(rel - predicted) < 0.05 * predicted
    # higher up the aliasing term is ~1e-21; what remains is the Euler-Maclaurin edge
    # term of the truncated window, O(h^2 z / R_edge^4) ~ 1e-8
    w = _wl(n, n, 1.0, 0.0, 0.0, ones, ones, ones, [[xc, xc, 8.0]])
    got = oracle.eval(w)[2, 0]
    omega = 4.0 * math.atan(a * b / (8.0 * math.sqrt(a * a + b * b + 64.0)))
    assert abs(got - omega / (2 * math.pi)) < 2e-8


# -- K-6 ---------------------------------------------------------------------
def _dipole_err(n, sel=None):
    w = config1(n)
    if sel is not None:
        w = w.subset(sel)
    B = oracle.eval(w)
    ref = np.array(dipole_field(w.x, w.y, w.z))
    return np.linalg.norm(B - ref, axis=0) / np.linalg.norm(ref, axis=0), w


def test_k6_buried_dipole_profile_and_convergence():
    err, w = _dipole_err(16)
    prof = err.reshape(8, 64).max(axis=1)
    tab = _read_table("k6_dipole_profile.txt")
    assert np.all(np.abs(prof - tab[:, 1]) <= 0.10 * tab[:, 1] + 5e-4)
    # widening the window about the dipole converges to the closed form
    e64, w64 = _dipole_err(64)
    assert e64[w64.z >= 2.0].max() <= 1.5e-3
    sel = np.arange(512)[::7]            # 74 points spread over all heights
    e256, w256 = _dipole_err(256, sel)
    assert e256[w256.z >= 3.0].max() <= 6e-6
    e1k, w1k = _dipole_err(1024, sel[::2])
    assert e1k[w1k.z >= 4.0].max() <= 3e-8
    assert e1k[w1k.z >= 4.0].max() < e256[w256.z >= 4.0].max() < e64[w64.z >= 4.0].max()


# -- K-7 ---------------------------------------------------------------------
def test_k7_helmholtz_invariant():
    """For fixed lambda the nodal sum u satisfies laplace(u) + lambda^2 u = 0 in z>0
    exactly (each term is -d/dz_i[cos(lam r)/r] h^2 B_k / 2 pi).  The 7-point Laplacian has
    an O(d^2) truncation error, removed here by one Richardson step."""
    w = random_boundary(12, 9, seed=1, npts=1)
    lam = 0.37
    p = np.array([5.3, 4.1, 2.6])

    def lap(d):
        offs = [np.zeros(3)] + [s * d * e for e in np.eye(3) for s in (1, -1)]
        pts = np.array([p + o for o in offs])
        ww = _wl(w.nx, w.ny, w.h, w.x0, w.y0, w.bx, w.by, w.bz, pts, np.full((3, 7), lam))
        B = oracle.eval(ww)
        return (B[:, 1:].sum(axis=1) - 6 * B[:, 0]) / (d * d), B[:, 0]

    l1, u = lap(0.04)
    l2, _ = lap(0.02)
    scale = np.abs(lam * lam * u).max()
    r1, r2 = l1 + lam * lam * u, l2 + lam * lam * u
    assert np.allclose(r1, 4.0 * r2, rtol=2e-3)                 # pure O(d^2) truncation
    assert np.all(np.abs((4 * l2 - l1) / 3 + lam * lam * u) <= 1e-6 * scale)
    # with a wrong lambda in the invariant it fails by orders of magnitude
    assert np.abs((4 * l2 - l1) / 3 + (1.1 * lam) ** 2 * u).max() > 1e-2 * scale


# -- K-8 ---------------------------------------------------------------------
def test_k8_symmetries():
    w = random_boundary(10, 7, seed=2, h=0.5, x0=-1.0, y0=2.0, npts=9)
    B = oracle.eval(w)
    # even in lambda, bit for bit
    assert np.array_equal(B, oracle.eval(w, lam=-w.lam))
    # linear in B0
    w2 = _wl(w.nx, w.ny, w.h, w.x0, w.y0, 2.5 * w.bx, -1.0 * w.by, 0.0 * w.bz,
             np.stack([w.x, w.y, w.z], 1), w.lam)
    B2 = oracle.eval(w2)
    assert np.allclose(B2[0], 2.5 * B[0], rtol=1e-14)
    assert np.allclose(B2[1], -B[1], rtol=1e-14)
    assert np.all(B2[2] == 0.0)
    # each component depends on its own lambda only (separability)
    lam3 = w.lam.copy(); lam3[1] *= 1.7
    B3 = oracle.eval(w, lam=lam3)
    assert np.array_equal(B3[0], B[0]) and np.array_equal(B3[2], B[2])
    assert not np.allclose(B3[1], B[1])
    # shifting the frame (x0, y0 and the points together)
    w4 = _wl(w.nx, w.ny, w.h, w.x0 + 3.0, w.y0 - 5.0, w.bx, w.by, w.bz,
             np.stack([w.x + 3.0, w.y - 5.0, w.z], 1), w.lam)
    assert np.allclose(oracle.eval(w4), B, rtol=1e-12)
    # 90 degree rotation of grid and points: (x, y) -> (-y, x)
    bx = w.bx.reshape(w.ny, w.nx); by = w.by.reshape(w.ny, w.nx); bz = w.bz.reshape(w.ny, w.nx)
    rot = lambda a: np.ascontiguousarray(a.T[:, ::-1])    # new[iy'=ix, ix'=ny-1-iy]
    w5 = _wl(w.ny, w.nx, w.h, -(w.y0 + w.ny * w.h), w.x0, rot(bx), rot(by), rot(bz),
             np.stack([-w.y, w.x, w.z], 1), w.lam)
    assert np.allclose(oracle.eval(w5), B, rtol=1e-12)
    # scaling lengths by s and lambda by 1/s leaves B unchanged (units, reading A-11)
    s = 3.0
    w6 = _wl(w.nx, w.ny, w.h * s, w.x0 * s, w.y0 * s, w.bx, w.by, w.bz,
             np.stack([w.x * s, w.y * s, w.z * s], 1), w.lam / s)
    assert np.allclose(oracle.eval(w6), B, rtol=1e-12)


# -- K-9 ---------------------------------------------------------------------
def _analytic_grad(w, p, lam):
    """dB_p/d(x_i,y_i,z_i) from d/dr[n(lam r)/r^3] = lam^2 cos(lam r)/r^2 - 3 n/r^4."""
    xk = w.x0 + (np.arange(w.nx) + 0.5) * w.h
    yk = w.y0 + (np.arange(w.ny) + 0.5) * w.h
    Yk, Xk = np.meshgrid(yk, xk, indexing="ij")
    dx, dy, z = (Xk - p[0]).ravel(), (Yk - p[1]).ravel(), p[2]
    r = np.sqrt(dx * dx + dy * dy + z * z)
    G = np.zeros((3, 3))
    c = w.h ** 2 / (2 * math.pi)
    for comp, b0 in enumerate((w.bx, w.by, w.bz)):
        l = abs(lam[comp])
        n = l * r * np.sin(l * r) + np.cos(l * r)
        dk = l * l * np.cos(l * r) / r ** 2 - 3 * n / r ** 4     # d/dr of n/r^3
        G[comp, 0] = c * np.sum(z * dk * (-dx / r) * b0)
        G[comp, 1] = c * np.sum(z * dk * (-dy / r) * b0)
        G[comp, 2] = c * np.sum((n / r ** 3 + z * dk * (z / r)) * b0)
    return G


def test_k9_forward_difference_stencil_vs_analytic_gradient():
    w = random_boundary(14, 11, seed=3, npts=4, zmin=1.5, zmax=5.0)
    errs = []
    for delta in (1e-3, 2.5e-4):
        res = oracle.residual(w, w.lam, oracle.Opts(delta=delta))
        worst = 0.0
        for i in range(w.M):
            G = _analytic_grad(w, (w.x[i], w.y[i], w.z[i]), w.lam[:, i])
            J = np.array([G[2, 1] - G[1, 2], G[0, 2] - G[2, 0], G[1, 0] - G[0, 1]])
            div = np.trace(G)
            scale = np.abs(G).max()
            worst = max(worst, np.abs(res["J"][:, i] - J).max() / scale,
                        abs(res["div"][i] - div) / scale)
            B = res["B"][:, i]
            f = np.linalg.norm(np.cross(J, B)) / (np.linalg.norm(J) * np.linalg.norm(B))
            g = abs(div) * (w.h / 6.0) / np.linalg.norm(B)
            assert abs(res["f"][i] - f) < 20 * delta
            assert abs(res["g"][i] - g) < 20 * delta * max(g, 1e-3)
            assert abs(res["phi"][i] - (res["f"][i] + res["g"][i])) < 1e-15
        errs.append(worst)
    assert errs[0] <= 5e-3                       # <= 5 delta / h
    assert errs[1] < 0.4 * errs[0]               # -> 0 linearly in delta


# -- K-10 --------------------------------------------------------------------
def test_k10_oracle_rounding_vs_mpmath():
    mp.mp.dps = 30
    w = random_boundary(16, 16, seed=4, npts=10)
    B = oracle.eval(w)
    for i in range(w.M):
        for comp, b0 in enumerate((w.bx, w.by, w.bz)):
            l = abs(w.lam[comp, i])
            tot = mp.mpf(0); mag = mp.mpf(0)
            for iy in range(w.ny):
                for ix in range(w.nx):
                    xk = w.x0 + (ix + 0.5) * w.h
                    yk = w.y0 + (iy + 0.5) * w.h
                    r = mp.sqrt((mp.mpf(xk) - w.x[i]) ** 2 + (mp.mpf(yk) - w.y[i]) ** 2
                                + mp.mpf(w.z[i]) ** 2)
                    t = (l * r * mp.sin(l * r) + mp.cos(l * r)) / r ** 3 * mp.mpf(float(b0[iy * w.nx + ix]))
                    tot += t; mag += abs(t)
            c = mp.mpf(w.z[i]) * w.h ** 2 / (2 * mp.pi)
            assert abs(mp.mpf(float(B[comp, i])) - c * tot) <= mp.mpf(1e-14) * c * mag


# -- S-1 ---------------------------------------------------------------------
def _rosen3(x):
    return (100.0 * (x[1] - x[0] * x[0]) ** 2 + (1.0 - x[0]) ** 2
            + 100.0 * (x[2] - x[1] * x[1]) ** 2 + (1.0 - x[1]) ** 2)


def _quad3(x):
    d0, d1, d2 = x[0] - 0.3, x[1] + 0.2, x[2] - 0.1
    return 3.0 * d0 * d0 + 0.5 * d1 * d1 + 2.0 * d2 * d2 + 0.7 * d0 * d1 - 0.4 * d1 * d2


def _abs3(x):   # non-smooth: forces contractions and shrinks
    return abs(x[0] - 0.1) + 2.0 * abs(x[1] + 0.3) + abs(x[0] * x[2]) + abs(x[2] - 0.2)


@pytest.mark.parametrize("fn,start,step", [(_rosen3, -1.2, 0.4), (_quad3, 0.05, 0.05),
                                           (_abs3, 0.05, 0.05), (_rosen3, 0.05, 0.05)])
def test_s1_nelder_mead_matches_scipy_iterate_by_iterate(fn, start, step):
    sim = np.full((4, 3), start)
    for j in range(3):
        sim[j + 1, j] += step
    maxiter = 150
    xtol, ftol = 1e-7, 1e-9
    mine = oracle.nm_generic(fn, sim, xtol, ftol, maxiter)
    ref = optimize.minimize(fn, sim[0], method="Nelder-Mead",
                            options={"initial_simplex": sim, "adaptive": False, "xatol": xtol,
                                     "fatol": ftol, "maxiter": maxiter + 1, "maxfev": 10 ** 6,
                                     "return_all": True})
    allvecs = np.array(ref.allvecs)
    # SciPy starts its counter at 1: nit = 1 + number of simplex updates performed
    assert mine["iters"] == ref.nit - 1
    assert mine["nfev"] == ref.nfev
    assert mine["trace"].shape == allvecs.shape
    # SciPy records allvecs[0] before its initial sort; compare the sorted sequence from 1 on
    assert np.allclose(mine["trace"][1:], allvecs[1:], rtol=0, atol=1e-15)
    assert fn(mine["trace"][0]) == min(fn(v) for v in sim)
    assert np.allclose(mine["simplex"], ref.final_simplex[0], rtol=0, atol=1e-15)
    assert np.allclose(mine["f"], ref.final_simplex[1], rtol=0, atol=1e-15)
    assert mine["status"] == (1 if ref.status == 0 else 2)


# -- S-4 ---------------------------------------------------------------------
def _numpy_eval(w, p, lam):
    xk = w.x0 + (np.arange(w.nx) + 0.5) * w.h
    yk = w.y0 + (np.arange(w.ny) + 0.5) * w.h
    Yk, Xk = np.meshgrid(yk, xk, indexing="ij")
    r = np.sqrt((Xk - p[0]) ** 2 + (Yk - p[1]) ** 2 + p[2] ** 2).ravel()
    out = []
    for comp, b0 in enumerate((w.bx, w.by, w.bz)):
        th = abs(lam[comp]) * r
        out.append(p[2] * w.h ** 2 / (2 * np.pi) * np.sum((th * np.sin(th) + np.cos(th)) / r ** 3 * b0))
    return np.array(out)


def _numpy_phi(w, p, lam, delta=1e-3, cell=1.0, w_g=1.0):
    d = delta * w.h
    p = np.asarray(p, float)
    B0 = _numpy_eval(w, p, lam)
    G = np.stack([(_numpy_eval(w, p + d * e, lam) - B0) / d for e in np.eye(3)], axis=1)
    J = np.array([G[2, 1] - G[1, 2], G[0, 2] - G[2, 0], G[1, 0] - G[0, 1]])
    f = np.linalg.norm(np.cross(J, B0)) / (np.linalg.norm(J) * np.linalg.norm(B0))
    g = abs(np.trace(G)) * (cell * w.h / 6.0) / np.linalg.norm(B0)
    return f + w_g * g, f, g, B0


def test_s4_brute_force_tiny_grid():
    w = random_boundary(4, 4, seed=5, npts=2, zmin=1.0, zmax=3.0)
    B = oracle.eval(w)
    res = oracle.residual(w, w.lam)
    for i in range(2):
        p = (w.x[i], w.y[i], w.z[i])
        assert np.allclose(B[:, i], _numpy_eval(w, p, w.lam[:, i]), rtol=1e-13)
        phi, f, g, B0 = _numpy_phi(w, p, w.lam[:, i])
        # forward differences amplify rounding by 1/delta
        assert abs(res["f"][i] - f) < 1e-9 and abs(res["g"][i] - g) < 1e-9
    # exhaustive lambda scan: the simplex result is no worse than the best scan node
    # reachable from its start (local method: compare with scan restricted to the box it searched)
    sol = oracle.solve_nm(w, oracle.Opts(use_eq12=0, maxiter=300))
    for i in range(2):
        p = (w.x[i], w.y[i], w.z[i])
        phi_star = _numpy_phi(w, p, sol["lam"][:, i])[0]
        assert abs(phi_star - sol["phi"][i]) < 1e-8
        assert abs(sol["f"][i] + sol["g"][i] - sol["phi"][i]) < 1e-15
        phi_start = _numpy_phi(w, p, np.full(3, 0.05 / w.h))[0]
        assert sol["phi"][i] <= phi_start + 1e-12
        # local optimality on a 21^3 scan of half-width 0.02/h around lambda*
        best = np.inf
        ax = np.linspace(-0.02, 0.02, 21) / w.h
        for a in ax:
            for b in ax:
                for c in ax:
                    best = min(best, _numpy_phi(w, p, sol["lam"][:, i] + np.array([a, b, c]))[0])
        assert sol["phi"][i] <= best + 5e-5


def test_solver_invalid_points_and_statuses():
    w = random_boundary(6, 6, seed=6, npts=4)
    z = w.z.copy(); z[1] = 0.0; z[2] = -1.0
    x = w.x.copy(); x[3] = np.nan
    sol = oracle.solve_nm(w, oracle.Opts(maxiter=5), x=x, z=z)
    assert list(sol["status"][1:]) == [3, 3, 3]
    assert np.all(np.isnan(sol["B"][:, 1:])) and np.all(np.isnan(sol["lam"][:, 1:]))
    assert sol["status"][0] in (0, 1, 2) and np.all(np.isfinite(sol["B"][:, 0]))
    assert sol["iters"][0] <= 5
    B = oracle.eval(w, x=x, z=z)
    assert np.all(np.isnan(B[:, 1:])) and np.all(np.isfinite(B[:, 0]))
    # M = 0 is a no-op
    assert oracle.eval(w, x=np.zeros(0), y=np.zeros(0), z=np.zeros(0), lam=np.zeros((3, 0))).shape == (3, 0)


# -- O-4 (GRID) ---------------------------------------------------------------
@pytest.mark.parametrize("analytic", [0, 1])
def test_grid_mode_brute_force_and_monotone(analytic):
    """O-4 with Eq. 13 differences and with the analytic gradient (O-5): the separable candidate
    assembly must equal a direct objective evaluation at every lattice triple."""
    w = random_boundary(5, 6, seed=8, npts=3, zmin=1.0, zmax=3.0)
    T = 4
    phis = []
    for nl in (1, 2, 3, 5):
        o = oracle.Opts(method=1, n_trial=T, n_level=nl, lam_max=0.4, use_eq12=0, analytic=analytic)
        sol = oracle.solve_grid(w, o)
        phis.append(sol["phi"].copy())
        # returned residual is the residual at the returned lambda
        res = oracle.residual(w, sol["lam"], o)
        assert np.allclose(res["phi"], sol["phi"], rtol=0, atol=1e-9)
        assert np.all(sol["iters"] == nl) and np.all(sol["status"] == 1)
    phis = np.array(phis)
    assert np.all(np.diff(phis, axis=0) <= 1e-15)      # incumbent never gets worse
    # level 0 is the exhaustive argmin over the T^3 lattice on [0, lam_max/h]
    ax = 0.4 / w.h * np.arange(T) / (T - 1)
    for i in range(w.M):
        best = np.inf
        for a in ax:
            for b in ax:
                for c in ax:
                    r = oracle.residual(w.subset([i]), np.array([[a], [b], [c]]), oracle.Opts(analytic=analytic))
                    best = min(best, r["phi"][0])
        assert abs(phis[0, i] - best) < 1e-9


# -- O-5: analytic gradient ------------------------------------
def _mp_field(w, comp, lam):
    """B_comp(x, y, z) of Eq. 6/16 as an mpmath function of the point (definition, 30 digits)."""
    b0 = (w.bx, w.by, w.bz)[comp]
    l = mp.mpf(abs(float(lam)))

    def f(x, y, z):
        tot = mp.mpf(0)
        for iy in range(w.ny):
            for ix in range(w.nx):
                xk = mp.mpf(w.x0) + (ix + mp.mpf(1) / 2) * mp.mpf(w.h)
                yk = mp.mpf(w.y0) + (iy + mp.mpf(1) / 2) * mp.mpf(w.h)
                r = mp.sqrt((xk - x) ** 2 + (yk - y) ** 2 + z ** 2)
                tot += (l * r * mp.sin(l * r) + mp.cos(l * r)) / r ** 3 * mp.mpf(float(b0[iy * w.nx + ix]))
        return z * mp.mpf(w.h) ** 2 / (2 * mp.pi) * tot
    return f


def test_g1_analytic_gradient_vs_mpmath_numerical_derivative():
    """The oracle's dB_p/dx_j against mpmath's numerical differentiation of the DEFINITION of B_p
    (no derivative formula is retyped here): a wrong sign, a dropped z-term of d/dz, or a
    transposed index fails it.  h != 1, shifted origin, lambda of both signs and lambda = 0."""
    mp.mp.dps = 30
    w = random_boundary(6, 5, seed=8, npts=3, h=0.5, x0=-1.0, y0=2.0, zmin=0.8, zmax=2.0)
    w.lam[:, 0] = 0.0
    w.lam[1, 1] = -w.lam[1, 1]
    B, G = oracle.gradient(w)
    assert np.allclose(B, oracle.eval(w), rtol=1e-14, atol=0)
    for i in range(w.M):
        pt = (mp.mpf(float(w.x[i])), mp.mpf(float(w.y[i])), mp.mpf(float(w.z[i])))
        for p in range(3):
            f = _mp_field(w, p, w.lam[p, i])
            for j in range(3):
                order = tuple(1 if q == j else 0 for q in range(3))
                ex = mp.diff(f, pt, order)
                scale = max(abs(G[p, :, i]).max(), 1e-300)
                assert abs(mp.mpf(float(G[p, j, i])) - ex) <= 1e-11 * scale, (i, p, j)


def test_g2_finite_differences_converge_to_the_analytic_gradient():
    """Eq. 13's forward differences of the oracle's own B approach the analytic gradient linearly
    in delta (pin K-9's statement, now between two oracle functions)."""
    w = random_boundary(14, 11, seed=3, npts=5, zmin=1.5, zmax=5.0)
    _, G = oracle.gradient(w)
    errs = []
    for d in (1e-2, 1e-3, 1e-4):
        B0 = oracle.eval(w)
        Gfd = np.empty_like(G)
        Gfd[:, 0] = (oracle.eval(w, x=w.x + d) - B0) / d
        Gfd[:, 1] = (oracle.eval(w, y=w.y + d) - B0) / d
        Gfd[:, 2] = (oracle.eval(w, z=w.z + d) - B0) / d
        errs.append(float((np.abs(Gfd - G).max(axis=(0, 1)) / np.abs(G).max(axis=(0, 1))).max()))
    assert errs[0] < 5e-2 and errs[1] < 0.2 * errs[0] and errs[2] < 0.2 * errs[1]


def test_g3_analytic_residual_and_solve_are_consistent_with_eq13():
    """residual(analytic=1) equals Eq. 8, 9, 14 applied to the analytic gradient, stays within
    O(delta) of the finite-difference residual, and the NM solve on it reaches an objective that is
    as good as the finite-difference solve's (cross-evaluated with the analytic objective)."""
    w = random_boundary(14, 11, seed=5, npts=6, zmin=1.5, zmax=5.0)
    ra = oracle.residual(w, w.lam, oracle.Opts(analytic=1))
    rf = oracle.residual(w, w.lam, oracle.Opts())
    B, G = oracle.gradient(w)
    J = np.array([G[2, 1] - G[1, 2], G[0, 2] - G[2, 0], G[1, 0] - G[0, 1]])
    assert np.array_equal(ra["J"], J) and np.array_equal(ra["div"], G[0, 0] + G[1, 1] + G[2, 2])
    nB = np.linalg.norm(B, axis=0)
    f = np.linalg.norm(np.cross(J.T, B.T), axis=1) / (np.linalg.norm(J, axis=0) * nB)
    assert np.allclose(ra["f"], f, rtol=1e-12) and np.allclose(ra["g"], np.abs(ra["div"]) * (w.h / 6.0) / nB, rtol=1e-12)
    assert np.abs(ra["f"] - rf["f"]).max() < 2e-2 and np.abs(ra["g"] - rf["g"]).max() < 2e-2 * max(1e-3, rf["g"].max())
    sa = oracle.solve_nm(w, oracle.Opts(analytic=1))
    sf = oracle.solve_nm(w, oracle.Opts())
    assert (sa["status"] != 3).all()
    cross = oracle.residual(w, sf["lam"], oracle.Opts(analytic=1))["phi"]
    assert np.all(sa["phi"] <= cross + 5e-3)          # both searches end in equally good minima
    assert np.all(sa["phi"] <= oracle.residual(w, np.full((3, w.M), 0.05 / w.h), oracle.Opts(analytic=1))["phi"] + 1e-15)


# -- O-6: 9-node element quadrature (Eq. 15) ------------------
def _nodes(n, h, c0):
    return c0 + (np.arange(n) + 0.5) * h


@pytest.mark.parametrize("nx,ny", [(7, 5), (6, 9), (8, 4), (3, 3)])
def test_q1_nine_node_staging_weights_and_interpolation(nx, ny):
    """Odd and even node counts.  (a) the weights of the Gauss-point sources sum to the integrated
    area (first to last node) in units of h^2; (b) nodal data that are globally biquadratic are
    reproduced exactly at every Gauss point (Lagrange interpolation on 3 x 3 nodes); (c) the rule
    integrates x^a y^b, a, b <= 2 (data) exactly: sum of staged values = closed-form integral."""
    h, x0, y0 = 0.5, -1.0, 2.0
    xn, yn = _nodes(nx, h, x0), _nodes(ny, h, y0)
    Y, X = np.meshgrid(yn, xn, indexing="ij")
    poly = lambda x, y: 1.5 - 0.7 * x + 0.3 * y + 0.2 * x * y - 0.4 * x * x + 0.1 * y * y + 0.05 * x * x * y * y
    one = np.ones(nx * ny)
    w = _wl(nx, ny, h, x0, y0, one, poly(X, Y).ravel(), (X * X * Y).ravel(), [[0.0, 0.0, 1.0]])
    xs, ys, s1, sp, sxy = oracle.q9_sources(w)
    nsx, nsy = 3 * (nx // 2), 3 * (ny // 2)
    assert xs.size == nsx and ys.size == nsy and s1.size == nsx * nsy
    assert np.all(np.diff(xs) > 0) and xs[0] > xn[0] and xs[-1] < xn[-1]
    assert abs(s1.sum() - (nx - 1) * (ny - 1)) < 1e-12 * nx * ny                       # (a)
    YS, XS = np.meshgrid(ys, xs, indexing="ij")
    wgt = s1.reshape(nsy, nsx)
    assert np.allclose(sp.reshape(nsy, nsx), wgt * poly(XS, YS), rtol=1e-12, atol=1e-13)   # (b)
    # (c) integral of x^2 y over [xn0, xn_last] x [yn0, yn_last], in units of h^2
    ex = (xn[-1] ** 3 - xn[0] ** 3) / 3.0 * (yn[-1] ** 2 - yn[0] ** 2) / 2.0 / (h * h)
    assert abs(sxy.sum() - ex) < 1e-12 * abs(ex)


def test_q2_nine_node_sum_equals_element_by_element_quadrature():
    """Eq. 15 written out independently: loop over elements, 3 x 3 Gauss points, shape functions,
    kernel of Eq. 6 at each Gauss point (NumPy), against oracle.eval on the staged sources."""
    import copy
    nx, ny, h, x0, y0 = 7, 9, 1.0, 0.0, 0.0
    w = random_boundary(nx, ny, seed=31, npts=5, h=h, x0=x0, y0=y0, zmin=1.0, zmax=4.0)
    w9 = copy.copy(w); w9.quad = 9
    B = oracle.eval(w9)
    g = np.array([-math.sqrt(0.6), 0.0, math.sqrt(0.6)]); gw = np.array([5, 8, 5]) / 9.0
    N = lambda t: np.array([t * (t - 1) / 2, 1 - t * t, t * (t + 1) / 2])
    data = [a.reshape(ny, nx) for a in (w.bx, w.by, w.bz)]
    for i in range(w.M):
        tot = np.zeros(3)
        for ey in range((ny - 1) // 2):
            for ex in range((nx - 1) // 2):
                for qy in range(3):
                    for qx in range(3):
                        xg = x0 + (2 * ex + 1.5) * h + g[qx] * h
                        yg = y0 + (2 * ey + 1.5) * h + g[qy] * h
                        r = math.sqrt((xg - w.x[i]) ** 2 + (yg - w.y[i]) ** 2 + w.z[i] ** 2)
                        Nq = np.outer(N(g[qy]), N(g[qx]))
                        for p in range(3):
                            th = abs(w.lam[p, i]) * r
                            val = (Nq * data[p][2 * ey:2 * ey + 3, 2 * ex:2 * ex + 3]).sum()
                            tot[p] += gw[qy] * gw[qx] * (th * math.sin(th) + math.cos(th)) / r ** 3 * val
        ref = w.z[i] * h * h / (2 * math.pi) * tot
        assert np.allclose(B[:, i], ref, rtol=1e-12, atol=0)


def test_q3_nine_node_agrees_with_the_nodal_rule_in_the_far_field():
    """Both discretisations converge to the same integral of a field that vanishes at the window
    edge: at z = 12 h and 24 h they agree to 5e-5 (the interpolant's flux differs from the midpoint sum by
    O((h/sigma)^4) for this sigma = 4 h Gaussian); near the boundary the two quadratures differ."""
    import copy
    n = 41
    c = (np.arange(n) + 0.5)
    Y, X = np.meshgrid(c, c, indexing="ij")
    bz = np.exp(-((X - 20.5) ** 2 + (Y - 20.5) ** 2) / (2 * 4.0 ** 2)).ravel()
    pts = [[18.3, 21.1, 12.0], [22.0, 19.0, 24.0], [20.5, 20.5, 1.0]]
    lam = np.array([[0.0, 0.1, 0.05]] * 3)
    w = _wl(n, n, 1.0, 0.0, 0.0, bz, 0.5 * bz, -bz, pts, lam)
    w9 = copy.copy(w); w9.quad = 9
    a, b = oracle.eval(w), oracle.eval(w9)
    rel = np.abs(a - b).max(axis=0) / np.abs(a).max(axis=0)
    assert rel[0] < 5e-5 and rel[1] < 5e-5              # what remains is the Simpson-vs-midpoint flux difference
    assert 1e-7 < rel[2] < 5e-2                         # z = h: the two quadratures differ


# -- margin (protocol P-4 rests on it) ---------------------------------------
def _table_objective(values):
    """Objective defined ONLY at the points one Nelder-Mead iteration can visit from the unit
    simplex V0 = 0, V1 = e1, V2 = e2, V3 = e3 (Phi = 10, 20, 30, 40): reflection (2/3, 2/3, -1),
    expansion (1, 1, -2), outside contraction (1/2, 1/2, -1/2), inside contraction (1/6, 1/6, 1/2),
    shrink vertices e_j / 2.  The geometry is O-3's formulas worked out by hand, not code."""
    pts = {"v0": (0, 0, 0), "v1": (1, 0, 0), "v2": (0, 1, 0), "v3": (0, 0, 1), "r": (2 / 3, 2 / 3, -1),
           "e": (1, 1, -2), "oc": (0.5, 0.5, -0.5), "ic": (1 / 6, 1 / 6, 0.5),
           "s1": (0.5, 0, 0), "s2": (0, 0.5, 0), "s3": (0, 0, 0.5)}
    vals = dict(v0=10.0, v1=20.0, v2=30.0, v3=40.0)
    vals.update(values)

    def fn(x):
        for k, p in pts.items():
            if np.allclose(x, p, atol=1e-12):
                return vals[k]       # KeyError = the driver visited a point this case does not define
        raise KeyError(tuple(x))
    return fn


@pytest.mark.parametrize("values,ftol,expect", [
    # reflection 9.7 < Phi_0 = 10 (gap 0.3, the closest) -> expansion 5 < 9.7 (gap 4.7); new order 5,10,20,30
    (dict(r=9.7, e=5.0), 1e-6, 0.3),
    # expansion not better than the reflection: 9.02 vs 9 (gap 0.02) -> reflection kept; order 9,10,20,30 (gap 1)
    (dict(r=9.0, e=9.02), 1e-6, 0.02),
    # 29.6: not < Phi_0 (19.6), < Phi_2 = 30 (gap 0.4) -> accepted; the new order 10,20,29.6,30 has the same gap
    (dict(r=29.6), 1e-6, 0.4),
    # 35: not < 30 (5), < Phi_3 = 40 (5) -> outside contraction 34.9 <= 35 (gap 0.1) accepted; order 10,20,30,34.9
    (dict(r=35.0, oc=34.9), 1e-6, 0.1),
    # 45 >= Phi_3 (5) -> inside contraction 39.95 < 40 (gap 0.05) accepted
    (dict(r=45.0, ic=39.95), 1e-6, 0.05),
    # inside contraction 41 not < 40 (gap 1) -> shrink; the new vertices 12, 12.25, 17 sort with gap 0.25
    (dict(r=45.0, ic=41.0, s1=12.0, s2=12.25, s3=17.0), 1e-6, 0.25),
    # the termination test max |Phi_j - Phi_0| = 30 against ftol = 29.99 is a decision too (gap 0.01)
    (dict(r=25.0), 29.99, 0.01),
])
def test_margin_is_the_closest_comparison_of_the_search(values, ftol, expect):
    """`margin` = the smallest |a - b| over every comparison a < b the search took (sorts, the ftol
    test, reflection / expansion / contraction decisions).  One iteration on a hand-built objective
    whose closest comparison is known.  The sort notes all six pairs; the smallest pair gap is always
    between neighbours of the sorted order, which the insertion sort compares directly, so this is the
    same number as the smallest gap over the comparisons actually executed."""
    sim = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1]], float)
    out = oracle.nm_generic(_table_objective(values), sim, 1e-9, ftol, 1)
    assert out["iters"] == 1
    assert out["margin"] == pytest.approx(expect, abs=1e-12)


def test_margin_of_the_point_solve_includes_the_eq12_tests():
    """orc_solve_nm also notes f vs eps_f and g vs eps_g (Eq. 12) at the best vertex: with eps_f set a
    hair below the f of the best initial vertex, the one iteration that follows has a margin of at most
    that hair (and exactly that hair when every other comparison is wider)."""
    w = random_boundary(9, 8, seed=12, npts=3, zmin=1.5, zmax=4.0)
    start = oracle.solve_nm(w, oracle.Opts(use_eq12=0, maxiter=0))     # best initial vertex, no iteration
    wide = oracle.solve_nm(w, oracle.Opts(use_eq12=0, maxiter=1))
    hair = 3e-9
    for i in range(w.M):
        o = oracle.Opts(use_eq12=1, maxiter=1, eps_f=float(start["f"][i]) - hair, eps_g=1e300)
        s = oracle.solve_nm(w.subset([i]), o)
        assert s["iters"][0] == 1 and s["status"][0] == 2          # the threshold was not met
        assert s["margin"][0] == pytest.approx(min(hair, wide["margin"][i]), rel=1e-6, abs=1e-15)
    assert (wide["margin"] > hair).any()


# -- O-4 (GRID): the refinement rule of levels >= 1 ---------------------------------------------
def _grid_by_the_book(w, i, T, L, lam_max, analytic, events):
    """DESIGN.md O-4 written out with the NumPy objective (no separability shortcut: every candidate
    triple is evaluated directly): window [lo, lo + W], trials lo + W t/(T-1), candidates = trials plus
    the incumbent (index T, levels >= 1), strict '<' in (t_x, t_y, t_z) order, next window of width
    2W/(T-1) centred on the argmin and clipped to [0, lam_max/h]."""
    p = np.array([w.x[i], w.y[i], w.z[i]])
    Lmax = lam_max / w.h
    lo, W, inc, best = np.zeros(3), Lmax, None, np.inf

    def phi_of(lam):
        if not analytic:
            return _numpy_phi(w, p, lam)[0]
        G, B0 = _analytic_grad(w, p, lam), _numpy_eval(w, p, lam)
        J = np.array([G[2, 1] - G[1, 2], G[0, 2] - G[2, 0], G[1, 0] - G[0, 1]])
        f = np.linalg.norm(np.cross(J, B0)) / (np.linalg.norm(J) * np.linalg.norm(B0))
        return f + abs(np.trace(G)) * (w.h / 6.0) / np.linalg.norm(B0)

    for lev in range(L):
        cands = [[lo[c] + W * t / (T - 1) for t in range(T)] + ([inc[c]] if inc is not None else [])
                 for c in range(3)]
        best, arg, second = np.inf, None, np.inf
        for tx, a in enumerate(cands[0]):
            for ty, b in enumerate(cands[1]):
                for tz, c in enumerate(cands[2]):
                    ph = phi_of(np.array([a, b, c]))
                    if ph < best:
                        second, best, arg = best, ph, (tx, ty, tz)
                    elif ph < second:
                        second = ph
        inc = np.array([cands[c][arg[c]] for c in range(3)])
        events["gap"] = min(events.get("gap", np.inf), second - best)
        events["incumbent_kept"] = events.get("incumbent_kept", 0) + sum(1 for c in range(3) if arg[c] == T)
        Wn = 2.0 * W / (T - 1)
        for c in range(3):
            l = inc[c] - 0.5 * Wn
            if l < 0.0:
                l = 0.0
                events["clip_lo"] = events.get("clip_lo", 0) + 1
            if l + Wn > Lmax:
                l = Lmax - Wn
                events["clip_hi"] = events.get("clip_hi", 0) + 1
            lo[c] = l
        W = Wn
    return inc, best


@pytest.mark.parametrize("T,lam_max,analytic", [(3, 0.4, 1), (4, 0.4, 1), (5, 0.03, 1), (4, 0.4, 0), (3, 0.03, 0)])
def test_grid_refinement_levels_by_brute_force(T, lam_max, analytic):
    """Pins levels 1-2 of O-4 (window recentring, clipping at 0 and at lam_max, the incumbent slot),
    not only level 0: orc_solve_grid after 1, 2 and 3 levels against the rule written out in NumPy.
    lam_max = 0.03 puts the optimum above the window, so the upper clip is exercised; lambda = 0
    winners exercise the lower one."""
    w = random_boundary(6, 5, seed=40 + T, npts=4, zmin=1.0, zmax=3.0)
    events = {}
    for L in (1, 2, 3):
        o = oracle.Opts(method=1, n_trial=T, n_level=L, lam_max=lam_max, use_eq12=0, analytic=analytic)
        sol = oracle.solve_grid(w, o)
        for i in range(w.M):
            ev = {}
            lam, phi = _grid_by_the_book(w, i, T, L, lam_max, analytic, ev)
            if ev["gap"] < (1e-10 if analytic else 1e-7):
                continue        # a near-tie of two candidates: the two evaluation orders may pick either
            for k, v in ev.items():
                events[k] = (min(events[k], v) if k == "gap" else events[k] + v) if k in events else v
            assert np.allclose(sol["lam"][:, i], lam, rtol=0, atol=1e-13 / w.h), (L, i)
            assert abs(sol["phi"][i] - phi) < (1e-12 if analytic else 1e-8)
    assert events.get("clip_lo", 0) + events.get("clip_hi", 0) > 0      # a window was clipped ...
    if lam_max < 0.1:
        assert events.get("clip_hi", 0) > 0                              # ... at lam_max
    assert "gap" in events                                               # some point was compared


# -- the oracle under ASan / UBSan ------------------------------------------------
def test_oracle_runs_clean_under_address_and_undefined_sanitizers(tmp_path):
    import shutil
    import subprocess
    if shutil.which("gcc") is None:
        pytest.skip("no gcc")
    exe = tmp_path / "orc_san"
    src = os.path.join(os.path.dirname(oracle.__file__), "sanitize_main.c")
    cc = ["gcc", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
          "-ffp-contract=off", "-fopenmp", "-o", str(exe), src, "-lm"]
    r = subprocess.run(cc, capture_output=True, text=True)
    if r.returncode != 0 and "sanitize" in r.stderr:
        pytest.skip("sanitizer runtime not installed: " + r.stderr.splitlines()[0])
    assert r.returncode == 0, r.stderr
    r = subprocess.run([str(exe)], capture_output=True, text=True,
                       env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1", OMP_NUM_THREADS="2"))
    assert r.returncode == 0, r.stdout + r.stderr
    assert "sanitize_main ok" in r.stdout


def test_k11_linear_force_free_field_is_recovered_with_lambda_equal_alpha():
    """Pins the PHYSICS of Eq. 6 with lambda != 0: for a constant-alpha force-free field whose
    boundary spectrum lies above alpha (every Fourier mode decays as exp(-sqrt(k^2 - alpha^2) z)), the boundary
    integral with lambda_x = lambda_y = lambda_z = alpha reproduces all three components of the field above the
    boundary, and lambda = 0 (the potential field of the same boundary) does not.  The reference is built here from
    the textbook mode solution (Nakagawa & Raadu 1972 form, derived from B = curl curl (P z) + alpha curl (P z) with
    (laplace + alpha^2) P = 0), checked to be force-free by finite differences, and evaluated by FFT; nothing of it
    comes from the oracle."""
    n, h, alpha = 512, 1.0, 0.3
    k0, sig = 0.8, 20.0
    c = (np.arange(n) - n // 2 + 0.5) * h                      # pixel centres, symmetric about 0
    Y, X = np.meshgrid(c, c, indexing="ij")
    bz0 = np.exp(-(X ** 2 + Y ** 2) / (2 * sig ** 2)) * (np.cos(k0 * X) + 0.5 * np.sin(0.9 * k0 * Y + 0.3 * k0 * X))
    kx = 2 * np.pi * np.fft.fftfreq(n, h)
    KY, KX = np.meshgrid(kx, kx, indexing="ij")
    K2 = KX ** 2 + KY ** 2
    Fz = np.fft.fft2(bz0)
    live = np.abs(Fz) > 1e-13 * np.abs(Fz).max()
    assert K2[live].min() > (1.2 * alpha) ** 2                 # every carried mode decays
    K2s = np.where(K2 > 0, K2, 1.0)
    L = np.sqrt(np.maximum(K2 - alpha ** 2, 0.0))
    Fz = np.where(live, Fz, 0.0)
    Fx = 1j * (alpha * KY - L * KX) / K2s * Fz
    Fy = -1j * (alpha * KX + L * KY) / K2s * Fz

    def at(z):
        d = np.exp(-L * z)
        return [np.real(np.fft.ifft2(F * d)) for F in (Fx, Fy, Fz)]

    # the reference really is force-free with this alpha: curl B = alpha B by central differences at z = 4
    e = 1e-3
    Bm, B0, Bp = at(4.0 - e), at(4.0), at(4.0 + e)
    ddz = [(p - m) / (2 * e) for p, m in zip(Bp, Bm)]
    spec = lambda f, K: np.real(np.fft.ifft2(1j * K * np.fft.fft2(f)))
    curl = [spec(B0[2], KY) - ddz[1], ddz[0] - spec(B0[2], KX), spec(B0[1], KX) - spec(B0[0], KY)]
    sc = max(np.abs(b).max() for b in B0)
    for cq, bq in zip(curl, B0):
        assert np.abs(cq - alpha * bq).max() <= 1e-6 * sc

    # boundary window: the central 256 x 256 pixels (the packet is 1e-9 of its peak at the window edge)
    m, o = 256, (n - 256) // 2
    win = (slice(o, o + m), slice(o, o + m))
    B00 = at(0.0)
    iy, ix = np.meshgrid(np.arange(o + 100, o + 156, 11), np.arange(o + 100, o + 156, 11), indexing="ij")
    pts = []
    ref = []
    for z in (3.0, 6.0, 12.0):
        Bz_ = at(z)
        for a, b in zip(iy.ravel(), ix.ravel()):
            pts.append((c[b], c[a], z))
            ref.append([Bz_[0][a, b], Bz_[1][a, b], Bz_[2][a, b]])
    pts = np.array(pts).T
    ref = np.array(ref).T
    w = Workload("lff_packet", m, m, h, c[o] - 0.5 * h, c[o] - 0.5 * h, B00[0][win].ravel(),
                           B00[1][win].ravel(), B00[2][win].ravel(), pts[0].copy(), pts[1].copy(), pts[2].copy())
    Ba = oracle.eval(w, lam=np.full((3, w.M), alpha))
    Bp0 = oracle.eval(w, lam=np.zeros((3, w.M)))
    scale = np.linalg.norm(ref, axis=0).max()
    err_a = np.linalg.norm(Ba - ref, axis=0).max() / scale
    err_0 = np.linalg.norm(Bp0 - ref, axis=0).max() / scale
    assert err_a <= 2e-6, err_a                                # lambda = alpha: the field, to quadrature accuracy
    assert err_0 >= 3e-2, err_0                                # lambda = 0: a different field
    # and the sign of the sin term / of alpha matters: lambda = 2 alpha is wrong as well
    err_2 = np.linalg.norm(oracle.eval(w, lam=np.full((3, w.M), 2 * alpha)) - ref, axis=0).max() / scale
    assert err_2 >= 3e-2, err_2


def test_k12_residual_on_the_constant_alpha_packet_gives_J_equal_alpha_B():
    """Pins the assembly of Eq. 14 (J = curl B: orientation and every entry), Eq. 8 (f) and Eq. 9 (g)
     on a field for which they are known: on the constant-alpha force-free packet of
    workloads/lff.py (the field of K-11, built there from the textbook mode solution and checked force-free by
    differences in tests/test_workloads.py; nothing of it comes from the oracle) with lambda_x = lambda_y =
    lambda_z = alpha, oracle.residual must return J = alpha B (closed form: alpha times the REFERENCE field, not
    the oracle's own B), div B = 0, f = 0 and g = 0, up to the first-order differences of Eq. 13 (delta = 1e-3 h)
    or, with the analytic gradient (O-5), up to the quadrature.  A J of the wrong sign gives |J - alpha B| =
    2 alpha |B|, two swapped entries of the curl or a transposed gradient give O(alpha |B|); alpha -> -alpha flips
    J.  With lambda = 0 or 2 alpha the same code reports what it should for a field that is NOT force-free with
    that boundary: J off alpha B by more than 20 %, f and g two orders of magnitude larger."""
    from workloads.lff import LFFPacket
    for alpha in (0.3, -0.3):
        w, ref = LFFPacket(alpha).workload()
        nB = np.linalg.norm(ref, axis=0)
        for analytic, tolJ, tolf, tolg in ((0, 6e-3, 5e-3, 2e-4), (1, 1e-4, 1e-4, 5e-6)):
            o = oracle.Opts(analytic=analytic)
            r = oracle.residual(w, np.full((3, w.M), alpha), o)
            assert (np.linalg.norm(r["B"] - ref, axis=0) / nB).max() <= 1e-5          # K-11 again, through O-2
            dJ = np.linalg.norm(r["J"] - alpha * ref, axis=0) / (abs(alpha) * nB)
            assert dJ.max() <= tolJ, (alpha, analytic, dJ.max())
            # orientation, said once more without a tolerance on the size: J . B has the sign of alpha everywhere
            assert np.all(np.sign((r["J"] * ref).sum(axis=0)) == np.sign(alpha))
            assert (np.abs(r["div"]) * w.h / nB).max() <= 6 * tolg
            assert r["f"].max() <= tolf and r["g"].max() <= tolg, (alpha, analytic, r["f"].max(), r["g"].max())
            assert np.all(r["f"] >= 0) and np.all(r["g"] >= 0)
            assert np.allclose(r["phi"], r["f"] + r["g"], rtol=0, atol=1e-15)         # reading A-7, w_g = 1
            for lam_wrong in (0.0, 2 * alpha):
                rw = oracle.residual(w, np.full((3, w.M), lam_wrong), o)
                dJw = np.linalg.norm(rw["J"] - alpha * ref, axis=0) / (abs(alpha) * nB)
                assert dJw.max() >= 0.2
                assert rw["f"].min() >= 0.02 and rw["f"].max() >= 0.2 and rw["g"].max() >= 1e-2
                assert np.all(rw["phi"] > r["phi"])
    # alpha -> -alpha mirrors the packet's transverse field and flips J (checked above through the sign of J . B);
    # and the three components of J are each pinned: rotate which component carries the error
    w, ref = LFFPacket(0.3).workload()
    r = oracle.residual(w, np.full((3, w.M), 0.3), oracle.Opts(analytic=1))
    for c in range(3):
        assert np.abs(r["J"][c] - 0.3 * ref[c]).max() <= 1e-4 * 0.3 * np.linalg.norm(ref, axis=0).max()
