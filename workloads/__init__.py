"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module holds NONE of the DBIE method's arithmetic (no Eq. 6 kernel, no
residuals, no optimiser): it only manufactures magnetograms, point sets and
lambda arrays.  It is the single piece of code shared by the CPU oracle
(`oracle/`) and the CUDA path (`paper_1306_1122_b200/`); neither of those two
imports the other.

The paper's real workload (SDO/HMI vector magnetogram of AR 11158, 300x300 px,
PAPER.md:177,225) is not available; the generators below take its shape (a few
compact kG spots, sheared transverse field along the inversion line, decaying
to ~0 at the window edge as PAPER.md:112 asks) and stand in for it.  The recipe
is stated in DESIGN.md section 4; seeds are 13061122 + config index.

Conventions (reading A-1): boundary arrays are row-major, x fastest,
pixel k = iy*nx + ix, pixel centre (x0 + (ix+1/2)h, y0 + (iy+1/2)h, 0).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

from .lowlou import LowLou

SEED_BASE = 13061122


@dataclasses.dataclass
class Workload:
    """One configuration: a boundary magnetogram plus evaluation points."""

    name: str
    nx: int
    ny: int
    h: float
    x0: float
    y0: float
    bx: np.ndarray          # (ny*nx,) float64
    by: np.ndarray
    bz: np.ndarray
    x: np.ndarray           # (M,) float64 evaluation points, z > 0
    y: np.ndarray
    z: np.ndarray
    lam: np.ndarray | None = None   # (3, M) float64 for eval-only configs
    extra: dict = dataclasses.field(default_factory=dict)
    quad: int = 0           # 0: one source per pixel centre (reading A-1); 9: 9-node elements (O-6)

    @property
    def N(self) -> int:
        return self.nx * self.ny

    @property
    def M(self) -> int:
        return int(self.x.shape[0])

    def subset(self, idx: np.ndarray) -> "Workload":
        """Same boundary, a subset of the points (used for oracle-sized parity)."""
        idx = np.asarray(idx)
        lam = None if self.lam is None else np.ascontiguousarray(self.lam[:, idx])
        return dataclasses.replace(
            self, x=np.ascontiguousarray(self.x[idx]), y=np.ascontiguousarray(self.y[idx]),
            z=np.ascontiguousarray(self.z[idx]), lam=lam)

    def seeded_subset(self, count: int, seed_offset: int = 0) -> tuple["Workload", np.ndarray]:
        """A seeded random subset of `count` points (sorted indices)."""
        rng = np.random.default_rng(SEED_BASE + 1000 + seed_offset)
        count = min(count, self.M)
        idx = np.sort(rng.choice(self.M, size=count, replace=False))
        return self.subset(idx), idx


def pixel_centres(n: int, h: float, origin: float) -> np.ndarray:
    return origin + (np.arange(n, dtype=np.float64) + 0.5) * h


def _grid_points(xs, ys, zs):
    """Volume points, x fastest, then y, then z."""
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    return (np.ascontiguousarray(X.ravel()), np.ascontiguousarray(Y.ravel()),
            np.ascontiguousarray(Z.ravel()))


# ----------------------------------------------------------------------------
# config 1: buried point dipole (closed form used as an external pin; A-15)
# ----------------------------------------------------------------------------
def dipole_field(x, y, z, pos=(8.0, 8.0, -4.0), m=(0.0, 0.0, 1.0)):
    """B(R) = [3 R (m.R)/R^5 - m/R^3] / (4 pi) of a point dipole at `pos`."""
    X = np.asarray(x, dtype=np.float64) - pos[0]
    Y = np.asarray(y, dtype=np.float64) - pos[1]
    Z = np.asarray(z, dtype=np.float64) - pos[2]
    R2 = X * X + Y * Y + Z * Z
    R = np.sqrt(R2)
    mR = m[0] * X + m[1] * Y + m[2] * Z
    c = 1.0 / (4.0 * math.pi)
    bx = c * (3.0 * X * mR / R**5 - m[0] / R**3)
    by = c * (3.0 * Y * mR / R**5 - m[1] / R**3)
    bz = c * (3.0 * Z * mR / R**5 - m[2] / R**3)
    return bx, by, bz


def config1(n: int = 16, centre_on_dipole: bool = True) -> Workload:
    """Potential-field sanity check: n x n window (default 16x16), unit spacing.

    With n != 16 the window is widened symmetrically about the dipole (same
    dipole, same points) for the convergence pin K-6.
    """
    h = 1.0
    x0 = y0 = 8.0 - 0.5 * n * h if centre_on_dipole else 0.0
    xs = pixel_centres(n, h, x0)
    ys = pixel_centres(n, h, y0)
    Y, X = np.meshgrid(ys, xs, indexing="ij")
    bx, by, bz = dipole_field(X.ravel(), Y.ravel(), np.zeros(n * n))
    px = 4.5 + np.arange(8, dtype=np.float64)
    pz = 1.0 + np.arange(8, dtype=np.float64)
    x, y, z = _grid_points(px, px, pz)
    lam = np.zeros((3, x.size))
    return Workload(f"cfg1_dipole_{n}x{n}", n, n, h, x0, y0, bx, by, bz, x, y, z, lam)


# ----------------------------------------------------------------------------
# config 2: Low & Lou analytic NLFFF
# ----------------------------------------------------------------------------
def config2(nb: int = 64, nz: int = 32, n: int = 1, m: int = 1, l: float = 0.3,
            Phi: float = math.pi / 4) -> Workload:
    ll = LowLou(n=n, m=m, l=l, Phi=Phi)
    h = 2.0 / nb
    x0 = y0 = -1.0
    xs = pixel_centres(nb, h, x0)
    Y, X = np.meshgrid(xs, xs, indexing="ij")
    bx, by, bz = ll.field(X.ravel(), Y.ravel(), np.zeros(nb * nb))
    scale = 1.0 / np.max(np.abs(bz))
    bx, by, bz = bx * scale, by * scale, bz * scale
    zs = (np.arange(nz, dtype=np.float64) + 1.0) * h
    x, y, z = _grid_points(xs, xs, zs)
    return Workload("cfg2_lowlou", nb, nb, h, x0, y0, bx, by, bz, x, y, z, None,
                    extra={"lowlou": ll, "scale": scale})


def lowlou_case2(nb: int = 192, nv: int = 64) -> Workload:
    """the paper's own validation case (Table 1): Low & Lou
    n = 3, m = 1, l = 0.3, Phi = 4 pi/5; the test region is [-1,1]^2 x (0,2] sampled by nv^3 points
    (pixel size h = 2/nv) and the bottom boundary is the nb x nb window centred on it ([-3,3]^2 for
    nb = 3 nv), "bottom boundary only".  Points: pixel centres x z = (k+1) h (reading A-14's
    convention; the paper does not say where its 64 layers sit).  Normalised to max|Bz| = 1."""
    ll = LowLou(n=3, m=1, l=0.3, Phi=4.0 * math.pi / 5.0)
    h = 2.0 / nv
    half = 0.5 * nb * h
    xb = pixel_centres(nb, h, -half)
    Y, X = np.meshgrid(xb, xb, indexing="ij")
    bx, by, bz = ll.field(X.ravel(), Y.ravel(), np.zeros(nb * nb))
    scale = 1.0 / np.max(np.abs(bz))
    xs = pixel_centres(nv, h, -1.0)
    zs = (np.arange(nv, dtype=np.float64) + 1.0) * h
    x, y, z = _grid_points(xs, xs, zs)
    return Workload("lowlou_case2", nb, nb, h, -half, -half, bx * scale, by * scale, bz * scale, x, y, z, None,
                    extra={"lowlou": ll, "scale": scale})


def figures_of_merit(B, b) -> dict:
    """The five figures of merit of Table 1 (the paper defers their definition
    to Schrijver et al. 2006): B exact, b reconstructed, both (3, M).  Evaluation metrics, not part
    of the method."""
    B = np.asarray(B, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    nB = np.linalg.norm(B, axis=0); nb_ = np.linalg.norm(b, axis=0)
    dot = np.sum(B * b, axis=0)
    d = np.linalg.norm(b - B, axis=0)
    return {"C_vec": float(dot.sum() / math.sqrt(np.sum(nB ** 2) * np.sum(nb_ ** 2))),
            "C_cs": float(np.mean(dot / (nB * nb_))),
            "E_n_prime": float(1.0 - d.sum() / nB.sum()),
            "E_m_prime": float(1.0 - np.mean(d / nB)),
            "eps": float(np.sum(nb_ ** 2) / np.sum(nB ** 2))}


# ----------------------------------------------------------------------------
# configs 3-5: Gaussian-spot active regions
# ----------------------------------------------------------------------------
def _spots_bz(n, centres, sigmas, amps):
    """Sum of Gaussian flux spots; negative amplitudes rescaled for zero net flux."""
    amps = np.array(amps, dtype=np.float64)
    sigmas = np.array(sigmas, dtype=np.float64)
    pos = amps > 0
    fpos = np.sum(amps[pos] * sigmas[pos] ** 2)
    fneg = -np.sum(amps[~pos] * sigmas[~pos] ** 2)
    amps[~pos] *= fpos / fneg
    c = np.arange(n, dtype=np.float64) + 0.5
    Y, X = np.meshgrid(c, c, indexing="ij")
    bz = np.zeros((n, n))
    for (cx, cy), s, a in zip(centres, sigmas, amps):
        bz += a * np.exp(-((X - cx) ** 2 + (Y - cy) ** 2) / (2.0 * s * s))
    return bz


def _potential_transverse(bz):
    """Transverse field of the potential extension of bz (FFT, periodic window)."""
    ny, nx = bz.shape
    kx = 2.0 * np.pi * np.fft.fftfreq(nx)
    ky = 2.0 * np.pi * np.fft.fftfreq(ny)
    KY, KX = np.meshgrid(ky, kx, indexing="ij")
    K = np.sqrt(KX * KX + KY * KY)
    K[0, 0] = 1.0
    bzh = np.fft.fft2(bz)
    bxh = -1j * KX / K * bzh
    byh = -1j * KY / K * bzh
    bxh[0, 0] = 0.0
    byh[0, 0] = 0.0
    return np.real(np.fft.ifft2(bxh)), np.real(np.fft.ifft2(byh))


def _sheared_region(n, centres, sigmas, amps, alpha0, rng, noise=10.0):
    bz = _spots_bz(n, centres, sigmas, amps)
    bx, by = _potential_transverse(bz)
    # shear concentrated on the polarity inversion line (Bz ~ 0), in px units
    dzy, dzx = np.gradient(bz)
    ell = float(np.mean(sigmas))
    alpha = alpha0 * np.exp(-(bz / 300.0) ** 2)
    bx = bx + alpha * ell * ell * dzy
    by = by - alpha * ell * ell * dzx
    bx = bx + rng.normal(0.0, noise, bz.shape)
    by = by + rng.normal(0.0, noise, bz.shape)
    bz = bz + rng.normal(0.0, noise, bz.shape)
    return bx.ravel().copy(), by.ravel().copy(), bz.ravel().copy()


def config3(n: int = 256, nsub: int = 128, nz: int = 64) -> Workload:
    """Synthetic bipolar active region, 0.5 Mm/px, 4 spots, alpha0 = 0.05/px."""
    rng = np.random.default_rng(SEED_BASE + 3)
    h = 0.5
    centres = rng.uniform(0.3 * n, 0.7 * n, size=(4, 2))
    sigmas = rng.uniform(3.0, 8.0, size=4) * (n / 256.0)
    amps = [1500.0, -1500.0, 1500.0, -1500.0]
    bx, by, bz = _sheared_region(n, centres, sigmas, amps, 0.05, rng)
    lo = (n - nsub) // 2
    xs = pixel_centres(n, h, 0.0)[lo:lo + nsub]
    zs = (np.arange(nz, dtype=np.float64) + 1.0) * h
    x, y, z = _grid_points(xs, xs, zs)
    return Workload("cfg3_bipolar", n, n, h, 0.0, 0.0, bx, by, bz, x, y, z, None)


def config4(n: int = 512, M: int = 1 << 20) -> Workload:
    """Kernel throughput sweep: fixed per-point per-component lambda."""
    rng = np.random.default_rng(SEED_BASE + 4)
    centres = rng.uniform(0.2 * n, 0.8 * n, size=(6, 2))
    sigmas = rng.uniform(6.0, 16.0, size=6) * (n / 512.0)
    amps = [1500.0, -1500.0, 1500.0, -1500.0, 1500.0, -1500.0]
    bz = _spots_bz(n, centres, sigmas, amps).ravel().copy()
    bx = rng.uniform(-500.0, 500.0, n * n)
    by = rng.uniform(-500.0, 500.0, n * n)
    x = rng.uniform(0.0, float(n), M)
    y = rng.uniform(0.0, float(n), M)
    z = rng.uniform(1.0, 0.5 * n, M)
    lam = rng.uniform(-0.2, 0.2, (3, M))
    return Workload("cfg4_sweep", n, n, 1.0, 0.0, 0.0, bx, by, bz, x, y, z, lam)


def config5(n: int = 1024, nsub: int = 256, nz: int = 128) -> Workload:
    """Large quadrupolar delta-spot region: 8 spots on an S-curve, alpha0 = 0.1/px."""
    rng = np.random.default_rng(SEED_BASE + 5)
    s = np.arange(8, dtype=np.float64)
    t = -1.0 + 2.0 * (s + 0.5) / 8.0
    sc = n / 1024.0
    cx = (512.0 + 300.0 * t) * sc
    cy = (512.0 + 120.0 * np.sin(np.pi * t) + np.where(s % 2 == 0, 60.0, -60.0)) * sc
    centres = np.stack([cx, cy], axis=1)
    sigmas = rng.uniform(12.0, 32.0, size=8) * sc
    amps = [1500.0 if i % 2 == 0 else -1500.0 for i in range(8)]
    bx, by, bz = _sheared_region(n, centres, sigmas, amps, 0.1, rng)
    lo = (n - nsub) // 2
    xs = pixel_centres(n, 1.0, 0.0)[lo:lo + nsub]
    zs = np.arange(nz, dtype=np.float64) + 1.0
    x, y, z = _grid_points(xs, xs, zs)
    return Workload("cfg5_delta", n, n, 1.0, 0.0, 0.0, bx, by, bz, x, y, z, None)


def random_boundary(nx: int, ny: int, seed: int, h: float = 1.0, x0: float = 0.0,
                    y0: float = 0.0, npts: int = 16, zmin: float = 1.0,
                    zmax: float = 8.0, lam_max: float = 0.2) -> Workload:
    """Small random boundary + random points, for unit tests and edge cases."""
    rng = np.random.default_rng(SEED_BASE + 100 + seed)
    N = nx * ny
    bx, by, bz = (rng.normal(0.0, 1.0, N) for _ in range(3))
    x = x0 + rng.uniform(0.0, nx * h, npts)
    y = y0 + rng.uniform(0.0, ny * h, npts)
    z = rng.uniform(zmin * h, zmax * h, npts)
    lam = rng.uniform(-lam_max / h, lam_max / h, (3, npts))
    return Workload(f"rand_{nx}x{ny}_s{seed}", nx, ny, h, x0, y0, bx, by, bz, x, y, z, lam)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}
