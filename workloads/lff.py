"""Constant-alpha (linear) force-free wave packet — INPUT GENERATOR only.

A field with curl B = alpha B, div B = 0 in z >= 0 whose every Fourier mode decays with height: the one
case in which the paper's pseudo-force-free factors are known in closed form (lambda_x = lambda_y =
lambda_z = alpha reproduces the field, PAPER.md:47-63 with lambda constant), so that Eq. 8, 9 and 14
 have known answers: J = alpha B, div B = 0, f = 0.  Pins K-11 / K-12 of
DESIGN.md section 3 and the GPU test of dbie_residual use it.  None of the DBIE arithmetic lives here.

Construction (the textbook mode solution, e.g. Nakagawa & Raadu 1972; from B = curl curl (P z^) +
alpha curl (P z^) with (laplace + alpha^2) P = 0): for each horizontal wave vector k with |k| > |alpha|,
    B^_z(k, z) = B^_z(k, 0) exp(-l z),  l = sqrt(k^2 - alpha^2),
    B^_x = i (alpha k_y - l k_x) / k^2 B^_z,   B^_y = -i (alpha k_x + l k_y) / k^2 B^_z.
B_z(x, y, 0) is a Gaussian-windowed pair of plane waves of wavenumber ~k0 > |alpha| on an n x n periodic
grid (the packet is 1e-9 of its peak at the edge of the central 256 x 256 window handed to DBIE).
tests/test_workloads.py checks curl B = alpha B by differences on what this returns.
"""
from __future__ import annotations

import numpy as np


class LFFPacket:
    def __init__(self, alpha: float = 0.3, n: int = 512, h: float = 1.0, k0: float = 0.8, sig: float = 20.0):
        self.alpha, self.n, self.h = float(alpha), n, h
        self.c = (np.arange(n) - n // 2 + 0.5) * h                  # pixel centres, symmetric about 0
        Y, X = np.meshgrid(self.c, self.c, indexing="ij")
        bz0 = np.exp(-(X ** 2 + Y ** 2) / (2 * sig ** 2)) * (np.cos(k0 * X) + 0.5 * np.sin(0.9 * k0 * Y + 0.3 * k0 * X))
        k = 2 * np.pi * np.fft.fftfreq(n, h)
        self.KY, self.KX = np.meshgrid(k, k, indexing="ij")
        K2 = self.KX ** 2 + self.KY ** 2
        Fz = np.fft.fft2(bz0)
        live = np.abs(Fz) > 1e-13 * np.abs(Fz).max()
        if not K2[live].min() > (1.2 * alpha) ** 2:
            raise ValueError("a carried mode does not decay: |k| <= 1.2 |alpha|")
        K2s = np.where(K2 > 0, K2, 1.0)
        self.L = np.sqrt(np.maximum(K2 - alpha ** 2, 0.0))
        self.Fz = np.where(live, Fz, 0.0)
        self.Fx = 1j * (alpha * self.KY - self.L * self.KX) / K2s * self.Fz
        self.Fy = -1j * (alpha * self.KX + self.L * self.KY) / K2s * self.Fz

    def at(self, z: float):
        """[Bx, By, Bz] on the n x n grid (row = y, column = x) at height z >= 0."""
        d = np.exp(-self.L * z)
        return [np.real(np.fft.ifft2(F * d)) for F in (self.Fx, self.Fy, self.Fz)]

    def workload(self, heights=(3.0, 6.0, 12.0), m: int = 256, lo: int = 100, hi: int = 156, stride: int = 11):
        """(Workload, ref): the central m x m window as the boundary and the grid points
        (lo:hi:stride)^2 of that window at each height; ref (3, M) = the field there."""
        from . import Workload
        n, h, c = self.n, self.h, self.c
        o = (n - m) // 2
        win = (slice(o, o + m), slice(o, o + m))
        B00 = self.at(0.0)
        iy, ix = np.meshgrid(np.arange(o + lo, o + hi, stride), np.arange(o + lo, o + hi, stride), indexing="ij")
        pts, ref = [], []
        for z in heights:
            Bz_ = self.at(z)
            for a, b in zip(iy.ravel(), ix.ravel()):
                pts.append((c[b], c[a], z))
                ref.append([Bz_[0][a, b], Bz_[1][a, b], Bz_[2][a, b]])
        pts = np.array(pts).T
        w = Workload(f"lff_packet_a{self.alpha:g}", m, m, h, c[o] - 0.5 * h, c[o] - 0.5 * h, B00[0][win].ravel().copy(),
                     B00[1][win].ravel().copy(), B00[2][win].ravel().copy(), pts[0].copy(), pts[1].copy(), pts[2].copy())
        return w, np.array(ref).T
