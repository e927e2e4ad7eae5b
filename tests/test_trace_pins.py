"""Pins of the tracing oracle (oracle/trace.py, reading T-1), CPU only.
None of them retypes the RK4 update: they check it against closed-form lines, a library integrator,
the order of convergence and the dipole field-line invariant r = L sin^2(theta)."""
import numpy as np
import pytest
from scipy import integrate

import oracle
from oracle import trace as otrace
import workloads

BIG = (-1e9, 1e9, -1e9, 1e9, -1e9, 1e9)


def _helix_field(c):
    return lambda P: np.stack([-P[1], P[0], np.full(P.shape[1], c)])


def _helix_exact(r0, s, c):
    """Line of v = (-y, x, c) through r0 in arc length: a helix of radius rho, pitch c / rho."""
    rho = np.hypot(r0[0], r0[1])
    w = 1.0 / np.sqrt(rho * rho + c * c)          # d(phi)/ds
    phi = np.arctan2(r0[1], r0[0]) + w * s
    return np.array([rho * np.cos(phi), rho * np.sin(phi), r0[2] + c * w * s])


def test_t1_helix_closed_form_and_fourth_order():
    """Arc-length RK4 on v = (-y, x, c): |v| is constant along a line, the exact line is a helix.
    Halving the step must divide the end-point error by ~16 (order 4)."""
    c, r0, S = 0.7, np.array([1.3, -0.4, 0.2]), 6.0
    errs = []
    for n in (24, 48, 96):
        path, npts, status = otrace.trace(_helix_field(c), r0[:, None], S / n, n, 1, BIG)
        assert npts[0] == n + 1 and status[0] == otrace.STOP_MAXSTEPS
        errs.append(np.linalg.norm(path[:, n, 0] - _helix_exact(r0, S, c)))
        # every stored point lies on the exact helix at its arc length (local check, not only the end)
        k = n // 3
        assert np.linalg.norm(path[:, k, 0] - _helix_exact(r0, S * k / n, c)) < 2 * errs[-1] + 1e-14
    assert errs[0] < 1e-4
    assert 12.0 < errs[0] / errs[1] < 20.0 and 12.0 < errs[1] / errs[2] < 20.0
    # against the field: the same helix backwards
    path, _, _ = otrace.trace(_helix_field(c), r0[:, None], S / 96, 96, -1, BIG)
    assert np.linalg.norm(path[:, 96, 0] - _helix_exact(r0, -S, c)) < 2 * errs[2]


def test_t2_against_a_library_integrator_on_the_lowlou_field():
    """Lines of the analytic Low & Lou field (the paper's validation field): the oracle's
    RK4 against scipy's DOP853 on dr/ds = B/|B| at tight tolerance."""
    w = workloads.config2()
    ll = w.extra["lowlou"]
    field = lambda P: np.array(ll.field(P[0], P[1], P[2]))
    seeds = np.array([[0.30, -0.25, 0.10], [0.05, 0.35, -0.30], [0.10, 0.15, 0.25]]).T.copy()
    seeds[2] = [0.10, 0.15, 0.25]
    S = 0.4

    def rhs(s, r):
        b = np.array(ll.field(np.array([r[0]]), np.array([r[1]]), np.array([r[2]]))).ravel()
        return b / np.linalg.norm(b)
    ref = [integrate.solve_ivp(rhs, (0.0, S), seeds[:, i], method="DOP853", rtol=1e-12, atol=1e-14,
                               t_eval=[S / 2, S]).y for i in range(seeds.shape[1])]
    errs = []
    for n in (40, 80):
        path, npts, status = otrace.trace(field, seeds, S / n, n, 1, BIG)
        assert np.all(npts == n + 1)
        e = 0.0
        for i in range(seeds.shape[1]):
            e = max(e, np.linalg.norm(path[:, n // 2, i] - ref[i][:, 0]), np.linalg.norm(path[:, n, i] - ref[i][:, 1]))
        errs.append(e)
    assert errs[0] < 1e-7 and errs[1] < errs[0] / 8.0, errs      # truncation error only, falling like ds^4


def test_t3_stop_conditions_and_bookkeeping():
    box = (0.0, 10.0, 0.0, 10.0, 0.0, 5.0)
    up = lambda P: np.stack([np.zeros(P.shape[1]), np.zeros(P.shape[1]), np.ones(P.shape[1])])
    seeds = np.array([[5.0, 5.0, 1.0],      # leaves through z_max = 5 after 8 steps of 0.5
                      [5.0, 5.0, 4.9],      # the first step's stage points leave at once
                      [11.0, 5.0, 1.0],     # seed outside the window
                      [5.0, 5.0, 0.0]]).T   # seed at z = z_min (the region is z > z_min)
    path, npts, status = otrace.trace(up, seeds, 0.5, 20, 1, box)
    assert list(npts) == [9, 1, 0, 0]
    assert list(status) == [otrace.STOP_LEFT] * 4
    assert np.allclose(path[2, :9, 0], 1.0 + 0.5 * np.arange(9)) and np.isnan(path[:, 9:, 0]).all()
    assert np.isnan(path[:, :, 2]).all()
    # downwards the same line stops just above z_min
    path, npts, status = otrace.trace(up, seeds[:, :1], 0.5, 20, -1, box)
    assert npts[0] == 2 and status[0] == otrace.STOP_LEFT and path[2, 1, 0] == 0.5
    # a field that vanishes (or is NaN) at a stage point stops the line with STOP_BADFIELD
    def dead_above_2(P):
        v = up(P)
        v[:, P[2] > 2.0] = 0.0
        return v
    path, npts, status = otrace.trace(dead_above_2, seeds[:, :1], 0.5, 20, 1, box)
    # steps 1 and 2 reach z = 1.5 and 2.0 (stages at <= 2.0); the second stage of step 3 sits at 2.25
    assert status[0] == otrace.STOP_BADFIELD and npts[0] == 3 and path[2, 2, 0] == 2.0
    nanf = lambda P: np.full_like(P, np.nan)
    _, npts, status = otrace.trace(nanf, seeds[:, :1], 0.5, 20, 1, box)
    assert status[0] == otrace.STOP_BADFIELD and npts[0] == 1
    # max_steps
    _, npts, status = otrace.trace(up, seeds[:, :1], 0.1, 7, 1, box)
    assert npts[0] == 8 and status[0] == otrace.STOP_MAXSTEPS


def test_t4_dipole_field_line_invariant():
    """BASELINE check 1 carried to the tracer: at lambda = 0 the DBIE field of a buried dipole's
    magnetogram is the dipole's field (up to window truncation, pin K-6), whose field lines are
    r = L sin^2(theta) about the dipole (theta from the moment axis).  L must stay constant along
    a traced line: 256x256 window, truncation <= 6e-6 for z >= 3."""
    w = workloads.config1(n=256)
    topts = otrace.TraceOpts(ds=0.25, max_steps=60, fixed_lam=(0.0, 0.0, 0.0), z_min=2.5)
    seeds = np.array([[9.5, 8.0, 6.0], [8.0, 6.0, 6.5], [10.0, 10.0, 6.0]]).T.copy()
    for direction in (1, -1):
        topts.direction = direction
        path, npts, status = otrace.trace_dbie(w, seeds, topts)
        for i in range(seeds.shape[1]):
            p = path[:, :npts[i], i]
            assert npts[i] >= 10
            X, Y, Z = p[0] - 8.0, p[1] - 8.0, p[2] + 4.0          # dipole at (8, 8, -4), moment along z
            R = np.sqrt(X * X + Y * Y + Z * Z)
            sin2 = (X * X + Y * Y) / (R * R)
            Lsh = R / sin2
            assert np.abs(Lsh / Lsh[0] - 1.0).max() < 2e-4, (direction, i, np.abs(Lsh / Lsh[0] - 1.0).max())
            # and the line moves: successive points are ds apart (arc-length parametrisation)
            d = np.linalg.norm(np.diff(p, axis=1), axis=0)
            assert np.allclose(d, 0.25, rtol=1e-3)
    # upwards (+B of a +z dipole above its axis region) z grows from the seed
    topts.direction = 1
    path, npts, _ = otrace.trace_dbie(w, seeds[:, :1], topts)
    assert path[2, npts[0] - 1, 0] != path[2, 0, 0]


def test_t5_current_lines_follow_J_and_solved_lambda_lines_follow_the_solved_field():
    """v = J (Eq. 14) at a fixed lambda, and v = B at the per-point solved lambda: the first step of the
    traced line is along the oracle's own J (or B) at the seed, to O(ds^2) of the line's curvature."""
    w, _ = workloads.config2().seeded_subset(4, seed_offset=1)
    seeds = np.stack([w.x, w.y, w.z + 4 * w.h])
    lam = np.full((3, 4), 0.08 / w.h)
    J = oracle.residual(w, lam, x=seeds[0], y=seeds[1], z=seeds[2])["J"]
    topts = otrace.TraceOpts(ds=0.05, max_steps=2, current=1, fixed_lam=(0.08 / w.h,) * 3)
    path, npts, status = otrace.trace_dbie(w, seeds, topts)
    assert np.all(npts == 3)
    step = (path[:, 1] - path[:, 0]) / (0.05 * w.h)
    assert np.abs(step - J / np.linalg.norm(J, axis=0)).max() < 2e-2
    s = oracle.solve_nm(w, x=seeds[0], y=seeds[1], z=seeds[2])
    path, npts, status = otrace.trace_dbie(w, seeds, otrace.TraceOpts(ds=0.05, max_steps=1))
    step = (path[:, 1] - path[:, 0]) / (0.05 * w.h)
    assert np.abs(step - s["B"] / np.linalg.norm(s["B"], axis=0)).max() < 5e-2
