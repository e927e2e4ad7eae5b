"""Low & Lou (1990) axisymmetric nonlinear force-free field — INPUT GENERATOR only.

Used to manufacture the boundary magnetogram of BASELINE.json config 2 (and the
analytic comparison field).  The paper validates against this benchmark
 but does not restate the construction; what follows is the
standard one, checked by its own self-test (tests/test_workloads.py: div B = 0
and curl B = alpha B by central differences, eigenvalue a^2 ~ 0.427 for
n=1, m=1).  None of the DBIE arithmetic lives here.

Construction.  In spherical coordinates (r, theta, phi) about a point source,
    B = [ (1/r) dA/dtheta  r^  -  dA/dr  theta^  +  Q  phi^ ] / (r sin theta),
    A = P(mu) / r^n,  mu = cos theta,  Q = a |A|^{1+1/n},
    (1 - mu^2) P'' + n(n+1) P + a^2 (1+n)/n  P |P|^{2/n} = 0,  P(+-1) = 0,
and alpha = dQ/dA = a (1+1/n) |A|^{1/n} sign(A).  The source sits at depth l
below the plane z = 0 and its axis is tilted by Phi about the y axis.
"""
from __future__ import annotations

import math

import numpy as np
from scipy.integrate import solve_ivp
from scipy.optimize import brentq


class LowLou:
    def __init__(self, n: int = 1, m: int = 1, l: float = 0.3, Phi: float = math.pi / 4,
                 dP0: float = 10.0):
        self.n, self.m, self.l, self.Phi, self.dP0 = n, m, l, Phi, dP0
        self._eps = 1e-7
        self.a2 = self._eigenvalue()
        self.a = math.sqrt(self.a2)
        self._sol = self._integrate(self.a2, dense=True)

    # -- the ODE for P(mu) ---------------------------------------------------
    def _integrate(self, a2, dense=False):
        n, eps = self.n, self._eps
        c = a2 * (1.0 + n) / n

        def rhs(mu, y):
            P, dP = y
            return [dP, -(n * (n + 1) * P + c * P * abs(P) ** (2.0 / n)) / (1.0 - mu * mu)]

        y0 = [self.dP0 * eps - 0.25 * n * (n + 1) * self.dP0 * eps * eps,
              self.dP0 - 0.5 * n * (n + 1) * self.dP0 * eps]
        return solve_ivp(rhs, (-1.0 + eps, 1.0 - eps), y0, method="DOP853",
                         rtol=1e-12, atol=1e-14, dense_output=dense)

    def _end_value(self, a2):
        s = self._integrate(a2)
        return s.y[0, -1] + self._eps * s.y[1, -1]

    def _eigenvalue(self):
        """a^2 of the m-th non-zero eigenvalue (m = number of sign changes' index)."""
        grid = np.concatenate([np.linspace(0.02, 2.0, 100), np.linspace(2.05, 40.0, 760)])
        prev_a2, prev_v, found = grid[0], self._end_value(grid[0]), 0
        for a2 in grid[1:]:
            v = self._end_value(a2)
            if prev_v * v < 0.0:
                found += 1
                if found == self.m:
                    return brentq(self._end_value, prev_a2, a2, xtol=1e-13, rtol=1e-13)
            prev_a2, prev_v = a2, v
        raise RuntimeError("Low & Lou eigenvalue not bracketed")

    def P(self, mu):
        mu = np.clip(mu, -1.0 + self._eps, 1.0 - self._eps)
        y = self._sol.sol(mu)
        return y[0], y[1]

    # -- the field -----------------------------------------------------------
    def _local(self, x, y, z):
        cP, sP = math.cos(self.Phi), math.sin(self.Phi)
        zz = np.asarray(z, dtype=np.float64) + self.l
        x = np.asarray(x, dtype=np.float64)
        return x * cP - zz * sP, np.asarray(y, dtype=np.float64), x * sP + zz * cP

    def field(self, x, y, z):
        """(Bx, By, Bz) at physical coordinates, arrays of equal shape."""
        n, a = self.n, self.a
        X, Y, Z = self._local(x, y, z)
        r = np.sqrt(X * X + Y * Y + Z * Z)
        mu = Z / r
        rho = np.sqrt(X * X + Y * Y)
        st = np.maximum(rho / r, 1e-300)
        cph = np.where(rho > 0, X / np.maximum(rho, 1e-300), 1.0)
        sph = np.where(rho > 0, Y / np.maximum(rho, 1e-300), 0.0)
        P, dP = self.P(mu)
        rn2 = r ** (n + 2)
        Br = -dP / rn2
        Bt = n * P / (rn2 * st)
        Bp = a * np.abs(P) ** (1.0 + 1.0 / n) / (rn2 * st)
        BX = Br * st * cph + Bt * mu * cph - Bp * sph
        BY = Br * st * sph + Bt * mu * sph + Bp * cph
        BZ = Br * mu - Bt * st
        cP, sP = math.cos(self.Phi), math.sin(self.Phi)
        return cP * BX + sP * BZ, BY, -sP * BX + cP * BZ

    def alpha(self, x, y, z):
        n, a = self.n, self.a
        X, Y, Z = self._local(x, y, z)
        r = np.sqrt(X * X + Y * Y + Z * Z)
        P, _ = self.P(Z / r)
        A = P / r ** n
        return a * (1.0 + 1.0 / n) * np.abs(A) ** (1.0 / n) * np.sign(A)
