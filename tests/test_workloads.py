"""Self-checks of the seeded input generators (workloads/) and the solver-level
pins S-2 / S-3 of DESIGN.md on an oracle-sized subset of config 2."""
import numpy as np
import pytest

import oracle
from workloads import CONFIGS, config2, config3, config4
from workloads.lowlou import LowLou


def test_lowlou_generator_is_force_free():
    """S-3 generator self-check: div B = 0, curl B = alpha B by central differences;
    first non-zero eigenvalue for n = 1 is a^2 ~ 0.4274 (Low & Lou quote 0.425)."""
    ll = LowLou(n=1, m=1, l=0.3, Phi=np.pi / 4)
    assert abs(ll.a2 - 0.42741) < 1e-4
    rng = np.random.default_rng(0)
    d = 1e-5
    for _ in range(6):
        q = np.array([rng.uniform(-0.8, 0.8), rng.uniform(-0.8, 0.8), rng.uniform(0.05, 1.0)])
        B = lambda v: np.array(ll.field(v[0], v[1], v[2]))
        G = np.stack([(B(q + d * e) - B(q - d * e)) / (2 * d) for e in np.eye(3)], axis=1)
        J = np.array([G[2, 1] - G[1, 2], G[0, 2] - G[2, 0], G[1, 0] - G[0, 1]])
        assert abs(np.trace(G)) < 1e-7 * np.abs(G).max()
        assert np.linalg.norm(J - ll.alpha(*q) * B(q)) < 1e-7 * np.linalg.norm(J)


def test_configs_are_seeded_and_shaped():
    w2 = config2()
    assert (w2.nx, w2.ny, w2.M) == (64, 64, 64 * 64 * 32)
    assert abs(np.abs(w2.bz).max() - 1.0) < 1e-12
    assert abs(w2.h - 2 / 64) < 1e-15 and w2.z.min() == w2.h and abs(w2.z.max() - 1.0) < 1e-12
    w3a, w3b = config3(), config3()
    assert np.array_equal(w3a.bx, w3b.bx) and np.array_equal(w3a.bz, w3b.bz)      # seeded
    assert (w3a.nx, w3a.M, w3a.h) == (256, 128 * 128 * 64, 0.5)
    assert 1200 < np.abs(w3a.bz).max() < 2500
    assert abs(w3a.bz.sum()) < 0.01 * np.abs(w3a.bz).sum()                       # net flux ~ 0
    edge = np.abs(w3a.bz.reshape(256, 256)[0]).max()
    assert edge < 100.0                                                           # -> 0 at the edge
    w4 = config4(M=4096)
    assert w4.lam.shape == (3, 4096) and np.abs(w4.lam).max() <= 0.2
    assert w4.z.min() >= 1.0 and w4.z.max() <= 256.0
    assert set(CONFIGS) == {1, 2, 3, 4, 5}


def test_s2_s3_lowlou_solve_invariants():
    """S-2: the search never ends above its start, status-0 points satisfy Eq. 12;
    S-3: the DBIE field is far more force-free than the potential (lambda = 0) field."""
    w = config2()
    s, _ = w.seeded_subset(48)
    o = oracle.Opts()
    sol = oracle.solve_nm(s, o)
    start = oracle.residual(s, np.full((3, s.M), o.lam0 / w.h), o)
    assert np.all(sol["phi"] <= start["phi"] + 1e-15)
    ok = sol["status"] == 0
    assert np.all(sol["f"][ok] <= o.eps_f) and np.all(sol["g"][ok] <= o.eps_g)
    assert np.all(sol["status"] <= 2) and np.all(sol["iters"] <= o.maxiter)
    assert np.all(sol["lam"] >= 0)
    pot = oracle.residual(s, np.zeros((3, s.M)), o)
    assert np.median(sol["f"]) < 0.05 and sol["f"].mean() < 0.3 * pot["f"].mean()
    # same order as the paper's <f_i> = 0.078, <g_i> = 6.7e-4 — loose sanity only
    assert sol["f"].mean() < 0.3 and sol["g"].mean() < 0.05
    # returned (B, f, g) are those of the returned lambda
    chk = oracle.residual(s, sol["lam"], o)
    assert np.allclose(chk["B"], sol["B"], rtol=1e-12, atol=0)
    assert np.allclose(chk["f"], sol["f"], atol=1e-9) and np.allclose(chk["g"], sol["g"], atol=1e-9)


def test_lowlou_case2_generator_and_figures_of_merit():
    """the n = 3, m = 1, Phi = 4 pi/5 field of the paper's Table 1 is force-free
    (same central-difference self-check), the workload has the paper's shape (192x192 boundary
    around a 64^3 region), and the five figures of merit are 1, 1, 1, 1, 1 for b = B and behave as
    defined for a scaled / rotated copy."""
    from workloads import lowlou_case2, figures_of_merit
    w = lowlou_case2()
    ll = w.extra["lowlou"]
    assert (w.nx, w.ny, w.M) == (192, 192, 64 ** 3) and abs(w.x0 + 3.0) < 1e-12 and abs(w.h - 2 / 64) < 1e-15
    assert abs(np.abs(w.bz).max() - 1.0) < 1e-12
    rng = np.random.default_rng(1)
    d = 1e-5
    for _ in range(4):
        q = np.array([rng.uniform(-0.8, 0.8), rng.uniform(-0.8, 0.8), rng.uniform(0.05, 1.0)])
        B = lambda v: np.array(ll.field(v[0], v[1], v[2]))
        G = np.stack([(B(q + d * e) - B(q - d * e)) / (2 * d) for e in np.eye(3)], axis=1)
        J = np.array([G[2, 1] - G[1, 2], G[0, 2] - G[2, 0], G[1, 0] - G[0, 1]])
        assert abs(np.trace(G)) < 1e-6 * np.abs(G).max()
        assert np.linalg.norm(J - ll.alpha(*q) * B(q)) < 1e-6 * np.linalg.norm(J)
    Bx = rng.normal(size=(3, 500))
    m = figures_of_merit(Bx, Bx)
    assert all(abs(v - 1.0) < 1e-12 for v in m.values())
    m2 = figures_of_merit(Bx, 2.0 * Bx)
    assert abs(m2["C_vec"] - 1) < 1e-12 and abs(m2["C_cs"] - 1) < 1e-12 and abs(m2["eps"] - 4) < 1e-12
    assert abs(m2["E_n_prime"]) < 1e-12 and abs(m2["E_m_prime"]) < 1e-12
    m3 = figures_of_merit(Bx, -Bx)
    assert abs(m3["C_vec"] + 1) < 1e-12 and abs(m3["E_n_prime"] + 1) < 1e-12


def test_lff_packet_generator_is_force_free_with_constant_alpha():
    """workloads/lff.py (the input of pins K-12 and of the GPU test of dbie_residual): curl B = alpha B and
    div B = 0 by differences (spectral in x, y; central in z) for both signs of alpha; the boundary window
    holds the packet (1e-9 of its peak at the edge); the points' reference values are the field there."""
    from workloads.lff import LFFPacket
    for alpha in (0.3, -0.3):
        p = LFFPacket(alpha)
        e = 1e-3
        Bm, B0, Bp = p.at(4.0 - e), p.at(4.0), p.at(4.0 + e)
        ddz = [(a - b) / (2 * e) for a, b in zip(Bp, Bm)]
        spec = lambda f, K: np.real(np.fft.ifft2(1j * K * np.fft.fft2(f)))
        curl = [spec(B0[2], p.KY) - ddz[1], ddz[0] - spec(B0[2], p.KX), spec(B0[1], p.KX) - spec(B0[0], p.KY)]
        sc = max(np.abs(b).max() for b in B0)
        for cq, bq in zip(curl, B0):
            assert np.abs(cq - alpha * bq).max() <= 1e-6 * sc
        assert np.abs(spec(B0[0], p.KX) + spec(B0[1], p.KY) + ddz[2]).max() <= 1e-6 * sc
        w, ref = p.workload()
        assert (w.nx, w.ny, w.M) == (256, 256, 108) and ref.shape == (3, 108)
        bz = w.bz.reshape(256, 256)
        assert max(np.abs(bz[0]).max(), np.abs(bz[:, 0]).max()) <= 1e-8 * np.abs(bz).max()
        # a point of the list sits on a pixel centre of the boundary grid, at the stated height
        i = 37
        ix = int(round((w.x[i] - w.x0) / w.h - 0.5)); iy = int(round((w.y[i] - w.y0) / w.h - 0.5))
        o = (p.n - 256) // 2
        assert abs(p.at(w.z[i])[2][o + iy, o + ix] - ref[2, i]) == 0.0
    with pytest.raises(ValueError):
        LFFPacket(0.9)                                           # modes with |k| <= 1.2 alpha would not decay
