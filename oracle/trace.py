"""ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Field-line and current-line tracing.  The paper shows field lines of the
reconstructed B and "current lines" of J = curl B (Eq. 14) in its Figs. 5-11
 but does not say how they were integrated.  Reading T-1: a line
through a seed r_0 is the solution of

    dr/ds = sigma * v(r) / |v(r)|,   v = B (field line) or v = J (current line),  sigma = +1 / -1,

in arc length s, integrated with the classical fourth-order Runge-Kutta scheme at a fixed step ds:

    k1 = u(r_n)            k2 = u(r_n + ds/2 k1)     k3 = u(r_n + ds/2 k2)     k4 = u(r_n + ds k3)
    r_{n+1} = r_n + ds/6 (k1 + 2 k2 + 2 k3 + k4),     u = sigma v / |v|.

v at a point is what the method gives there and nowhere else is anything interpolated: B from the
per-point lambda solve (O-3), or from Eq. 6 at a fixed lambda triple (O-1); J from the residual
(O-2) at that lambda.  A line stops when a stage point or the new point leaves the region
z > z_min, x0 <= x <= x0 + nx h, y0 <= y <= y0 + ny h, z <= z_max (status 1), when v is zero or
not finite at a stage (status 2), or after max_steps steps (status 0).  The last accepted point
is kept; nothing beyond it is written.

This is the algorithm written out step by step in NumPy, one stage at a time for all lines;
`field` may be any callable (pins use analytic fields), `dbie_field` wraps the oracle's own
solve / eval / residual.  It shares no code with paper_1306_1122_b200/.
"""
from __future__ import annotations

import dataclasses

import numpy as np

STOP_MAXSTEPS, STOP_LEFT, STOP_BADFIELD = 0, 1, 2


@dataclasses.dataclass
class TraceOpts:
    ds: float = 0.5            # step in arc length, as a FRACTION of h
    max_steps: int = 100
    direction: int = 1         # +1 along v, -1 against
    current: int = 0           # 0: v = B (field lines); 1: v = J (current lines, Eq. 14)
    fixed_lam: tuple | None = None   # None: lambda from the per-point solve; else a constant triple (units 1/length)
    z_min: float = 0.0         # region, z in fractions of h
    z_max: float = 1e300


def _inside(p, box):
    x0, x1, y0, y1, z0, z1 = box
    return (p[0] >= x0) & (p[0] <= x1) & (p[1] >= y0) & (p[1] <= y1) & (p[2] > z0) & (p[2] <= z1)


def trace(field, seeds, ds_abs: float, max_steps: int, direction: int, box):
    """RK4 in arc length for all seeds at once.  field(P) -> V: (3, n) -> (3, n) (NaN allowed).
    Returns path (3, max_steps + 1, L) (NaN past the end), npts (L,), status (L,)."""
    seeds = np.asarray(seeds, dtype=np.float64)
    L = seeds.shape[1]
    path = np.full((3, max_steps + 1, L), np.nan)
    npts = np.zeros(L, dtype=np.int32)
    status = np.full(L, STOP_MAXSTEPS, dtype=np.int32)
    r = seeds.copy()
    alive = _inside(r, box) & np.isfinite(r).all(axis=0)
    status[~alive] = STOP_LEFT
    path[:, 0, alive] = r[:, alive]
    npts[alive] = 1

    def unit(P, idx):
        """u = direction * v/|v| at the points P of the lines idx; ok = finite and non-zero."""
        V = np.asarray(field(P), dtype=np.float64)
        n = np.sqrt(V[0] * V[0] + V[1] * V[1] + V[2] * V[2])
        ok = np.isfinite(n) & (n > 0.0)
        with np.errstate(invalid="ignore", divide="ignore"):
            U = direction * V / n
        return U, ok

    for step in range(max_steps):
        idx = np.where(alive)[0]
        if idx.size == 0:
            break
        rn = r[:, idx]
        ks = []
        P = rn
        good = np.ones(idx.size, dtype=bool)       # still integrating this step
        why = np.zeros(idx.size, dtype=np.int32)
        for stage in range(4):
            ins = _inside(P, box)
            why[good & ~ins] = STOP_LEFT
            good &= ins
            U, ok = unit(np.where(good, P, rn), idx)   # stopped lines are evaluated at r_n (ignored)
            why[good & ~ok] = STOP_BADFIELD
            good &= ok
            ks.append(U)
            if stage < 3:
                c = 0.5 * ds_abs if stage < 2 else ds_abs
                P = rn + c * U
        rnew = rn + (ds_abs / 6.0) * (ks[0] + 2.0 * ks[1] + 2.0 * ks[2] + ks[3])
        ins = _inside(rnew, box) & np.isfinite(rnew).all(axis=0)
        why[good & ~ins] = STOP_LEFT
        good &= ins
        done = idx[~good]
        status[done] = why[~good]
        alive[done] = False
        keep = idx[good]
        r[:, keep] = rnew[:, good]
        path[:, step + 1, keep] = rnew[:, good]
        npts[keep] = step + 2
    return path, npts, status


def region(wl, topts: TraceOpts):
    return (wl.x0, wl.x0 + wl.nx * wl.h, wl.y0, wl.y0 + wl.ny * wl.h, topts.z_min * wl.h, topts.z_max * wl.h)


def dbie_field(wl, topts: TraceOpts, sopts=None):
    """v(P) from the oracle's own DBIE functions: B or J at the solved (or fixed) lambda."""
    import oracle

    def f(P):
        n = P.shape[1]
        if topts.fixed_lam is not None:
            lam = np.repeat(np.asarray(topts.fixed_lam, dtype=np.float64)[:, None], n, axis=1)
            if not topts.current:
                return oracle.eval(wl, x=P[0], y=P[1], z=P[2], lam=lam)
            return oracle.residual(wl, lam, sopts, x=P[0], y=P[1], z=P[2])["J"]
        s = oracle.solve_nm(wl, sopts, x=P[0], y=P[1], z=P[2])
        if not topts.current:
            return s["B"]
        J = oracle.residual(wl, np.where(np.isfinite(s["lam"]), s["lam"], 0.0), sopts, x=P[0], y=P[1], z=P[2])["J"]
        J[:, s["status"] == 3] = np.nan
        return J
    return f


def trace_dbie(wl, seeds, topts: TraceOpts | None = None, sopts=None):
    """Lines of the DBIE field of workload `wl` through `seeds` (3, L)."""
    topts = topts or TraceOpts()
    return trace(dbie_field(wl, topts, sopts), seeds, topts.ds * wl.h, topts.max_steps, topts.direction,
                 region(wl, topts))
