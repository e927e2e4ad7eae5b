"""GPU parity: the CUDA path (through the C ABI, libdbie_b200.so) against the CPU oracle on the
same seeded inputs.  Tolerances (BASELINE.json north_star; derivation in DESIGN.md section 8):
  B      : max_i ||dB_i|| / ||B_i||  <= 1e-9 over points with ||B_i|| >= 1e-6 max ||B||
  lambda : | |lam|_gpu - |lam|_orc | * h <= 1e-6 with identical status and iteration count on >= 99 %
           of the valid points of every solve batch (measured: 100 %; samples below 150 points may hold one
           fork); every other point must be an explained fork: oracle margin < 1e-7 (protocol P-4)
  f, g   : 1e-6 absolute
"""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

TOL_B = 1e-9
TOL_LAM = 1e-6
TOL_FG = 1e-6
MARGIN_STABLE = 1e-7


@pytest.fixture(scope="module")
def dbie():
    import torch
    assert torch.cuda.is_available()
    import paper_1306_1122_b200 as d
    d.load()     # raises if the CUDA library is missing: no fallback
    return d


def vec_relerr(B, R, floor=1e-6):
    n = np.linalg.norm(R, axis=0)
    keep = n >= floor * n.max()
    e = np.linalg.norm(B - R, axis=0)
    return float((e[keep] / n[keep]).max()), int((~keep).sum())


def gpu_eval(d, wl):
    with d.DBIE.from_workload(wl) as ctx:
        dw = d.to_device(wl)
        return ctx.eval(dw.x, dw.y, dw.z, dw.lam).cpu().numpy()


# ---------------------------------------------------------------------------- eval ---------
def test_config1_dipole_eval_matches_oracle_and_closed_form(dbie):
    """BASELINE configs[0]: lambda = 0, 16x16 window, 8x8x8 points; GPU == oracle to 1e-9 and the
    truncation-error profile vs the closed-form dipole is the one pinned in tests/golden."""
    w = workloads.config1()
    B = gpu_eval(dbie, w)
    R = oracle.eval(w)
    err, dropped = vec_relerr(B, R)
    assert err <= TOL_B and dropped == 0
    ex = np.array(workloads.dipole_field(w.x, w.y, w.z))
    rel = np.linalg.norm(B - ex, axis=0) / np.linalg.norm(ex, axis=0)
    prof = [rel[np.isclose(w.z, zz)].max() for zz in range(1, 9)]
    gold = np.loadtxt("tests/golden/k6_dipole_profile.txt")[:, 1]
    assert np.all(np.abs(np.array(prof) - gold) <= 0.1 * gold)


@pytest.mark.parametrize("nx,ny", [(1, 1), (1, 7), (7, 1), (17, 33), (513, 3), (3, 513), (1030, 2),
                                   (64, 64), (600, 5), (512, 4), (1024, 3), (2049, 1)])
def test_eval_ragged_boundaries(dbie, nx, ny):
    """Tile edges: one pixel, single rows/columns, widths just above the 512-pixel tile, odd tails;
    37 points (not a multiple of anything), h != 1, shifted origin, lambda of both signs."""
    w = workloads.random_boundary(nx, ny, seed=nx * 7 + ny, npts=37, h=0.5, x0=-1.0, y0=2.0)
    w.lam[:, 0] = 0.0
    w.lam[1, 1] = -w.lam[1, 1]
    err, _ = vec_relerr(gpu_eval(dbie, w), oracle.eval(w))
    assert err <= TOL_B


def test_eval_config4_first_points_fp64(dbie):
    """BASELINE configs[3] at full boundary size (512x512), first 1536 points: spans 3 work blocks
    with a ragged tail of the register-blocked mapping."""
    w = workloads.config4()
    sub = w.subset(np.arange(1536))
    err, dropped = vec_relerr(gpu_eval(dbie, sub), oracle.eval(sub))
    assert err <= TOL_B, err
    assert dropped == 0


def test_eval_config4_full_size_sampled(dbie):
    """Full M = 1,048,576 in the launch configuration bench.py times; 192 sampled outputs are
    recomputed one by one by the oracle; plus properties that hold at any size."""
    import torch
    w = workloads.config4()
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        B = ctx.eval(dw.x, dw.y, dw.z, dw.lam)
        B2 = ctx.eval(dw.x, dw.y, dw.z, dw.lam)
        assert torch.equal(B, B2)                      # run-to-run bitwise reproducible
        Bneg = ctx.eval(dw.x, dw.y, dw.z, -dw.lam)
        assert torch.equal(B, Bneg)                    # even in lambda (reading A-3), bit for bit
        assert bool(torch.isfinite(B).all())
        c = ctx.counters()
        assert c["interactions"] == float(w.M) * w.N
        # a result does not depend on the batch it was computed in (canonical chunk sums)
        idx = torch.arange(5000, 5000 + 777, device="cuda")
        Bs = ctx.eval(dw.x[idx].contiguous(), dw.y[idx].contiguous(), dw.z[idx].contiguous(),
                      dw.lam[:, idx].contiguous())
        assert torch.equal(Bs, B[:, idx])
        B = B.cpu().numpy()
    sub, idx = w.seeded_subset(192)
    err, _ = vec_relerr(B[:, idx], oracle.eval(sub))
    assert err <= TOL_B, err


def test_eval_reduced_sincos_flag_measured_error(dbie):
    """DBIE_EVAL_REDUCED_SINCOS (reading A-12: eval only, never the solver): sin/cos of the reduced argument
    with one coefficient fewer each (approximation error 3e-13).  Measured here on BASELINE configs[3]'s
    boundary and on config 2's: B must stay within the same 1e-9 as the full kernel, the solver must be
    untouched by the flag (bit-identical results), and the flag must really change the eval arithmetic."""
    import torch
    w = workloads.config4()
    sub, _ = w.seeded_subset(1024, seed_offset=3)
    ref = oracle.eval(sub)
    with dbie.DBIE.from_workload(sub, reduced_sincos=True) as ctx:
        dw = dbie.to_device(sub)
        Br = ctx.eval(dw.x, dw.y, dw.z, dw.lam).cpu().numpy()
    Bf = gpu_eval(dbie, sub)
    err_r, _ = vec_relerr(Br, ref)
    err_f, _ = vec_relerr(Bf, ref)
    print(f"reduced sincos: max |dB|/|B| = {err_r:.2e} (full kernel: {err_f:.2e})")
    assert err_r <= TOL_B and err_f <= TOL_B
    assert not np.array_equal(Br, Bf)
    w2, _ = workloads.config2().seeded_subset(64, seed_offset=11)
    with dbie.DBIE.from_workload(w2, reduced_sincos=True) as c1, dbie.DBIE.from_workload(w2) as c0:
        dw = dbie.to_device(w2)
        s1, s0 = c1.solve(dw.x, dw.y, dw.z), c0.solve(dw.x, dw.y, dw.z)
        for k in ("B", "lam", "f", "g", "iters", "status"):
            assert torch.equal(s1[k], s0[k]), k


def test_eval_edge_cases(dbie):
    import torch
    w = workloads.random_boundary(20, 12, seed=3, npts=9)
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        # M = 0 is a no-op
        e = torch.empty(0, dtype=torch.float64, device="cuda")
        out = ctx.eval(e, e, e, torch.empty((3, 0), dtype=torch.float64, device="cuda"))
        assert out.shape == (3, 0)
        # invalid points give NaN without failing the call; the others are untouched
        z = dw.z.clone(); z[2] = 0.0; z[5] = -1.0
        lam = dw.lam.clone(); lam[1, 7] = float("nan")
        B = ctx.eval(dw.x, dw.y, z, lam).cpu().numpy()
        good = ctx.eval(dw.x, dw.y, dw.z, dw.lam).cpu().numpy()
        bad = [2, 5, 7]
        assert np.isnan(B[:, bad]).all()
        ok = [i for i in range(9) if i not in bad]
        assert np.array_equal(B[:, ok], good[:, ok])
        # the host-pointer entry point gives the same bits as the device-pointer one
        Bh = ctx.eval_host(w.x, w.y, w.z, w.lam)
        assert np.array_equal(Bh, good)
        # wrong dtype / device are rejected by the binding
        with pytest.raises(TypeError):
            ctx.eval(dw.x.float(), dw.y, dw.z, dw.lam)
    # the oracle treats the same points as invalid
    wb = w.subset(np.arange(9)); wb.z[2] = 0.0
    assert np.isnan(oracle.eval(wb)[:, 2]).all()


def test_blocks_of_invalid_points_do_not_change_the_others(dbie):
    """Whole 256- (128-) point blocks of invalid points (what dbie_trace hands over for stopped lines: z = -1) and
    invalid stragglers inside live blocks: those outputs are NaN, and every other point keeps its bits, in dbie_eval,
    dbie_eval_noalloc and dbie_residual (both gradients)."""
    import torch
    w = workloads.random_boundary(96, 80, seed=21, npts=1500, h=0.7)
    dead = np.zeros(w.M, dtype=bool)
    dead[256:1024] = True                       # three whole eval blocks (six residual blocks)
    dead[[3, 1100, 1499]] = True                # and stragglers inside live blocks
    z = w.z.copy(); z[dead] = -1.0; z[300] = np.nan; z[301] = 0.0
    with dbie.DBIE.from_workload(w) as ctx:
        d = dbie.to_device(w)
        dz = torch.from_numpy(z).cuda()
        ref = ctx.eval(d.x, d.y, d.z, d.lam)
        B = ctx.eval(d.x, d.y, dz, d.lam)
        assert bool(torch.isnan(B[:, dead]).all()) and torch.equal(B[:, ~dead], ref[:, ~dead])
        rref = ctx.residual(d.x, d.y, d.z, d.lam)
        for an in (0, 1):
            o = dbie.default_opts(analytic=an)
            rr = ctx.residual(d.x, d.y, d.z, d.lam, o)
            r = ctx.residual(d.x, d.y, dz, d.lam, o)
            for k in ("B", "J"):
                assert bool(torch.isnan(r[k][:, dead]).all()) and torch.equal(r[k][:, ~dead], rr[k][:, ~dead])
            for k in ("f", "g", "div", "phi"):
                assert bool(torch.isnan(r[k][dead]).all()) and torch.equal(r[k][~dead], rr[k][~dead])
        # everything invalid: nothing to sum at all
        allbad = ctx.eval(d.x, d.y, -d.z, d.lam)
        assert bool(torch.isnan(allbad).all())
        out = torch.empty_like(ref)
        ctx.eval_noalloc(d.x, d.y, dz, d.lam, out)
        assert torch.equal(out[:, ~dead], ref[:, ~dead]) and bool(torch.isnan(out[:, dead]).all())


def test_eval_potential_field_fast_path_is_bit_identical(dbie):
    """Points with lambda = 0 in all three components take a loop without sincos (n(0) = 1 exactly).  Their
    result must equal, bit for bit, what the general loop gives: lambda = 1e-300 r underflows theta to a
    value whose n(theta) is exactly 1 as well, but takes the general path.  Mixed warps included."""
    import torch
    w = workloads.random_boundary(150, 90, seed=41, npts=700, h=0.5, zmin=0.5, zmax=40.0)
    lam0 = np.zeros((3, w.M))
    lam_tiny = np.full((3, w.M), 1e-300)
    lam_mixed = lam0.copy(); lam_mixed[:, ::2] = w.lam[:, ::2]
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        ev = lambda l: ctx.eval(dw.x, dw.y, dw.z, torch.from_numpy(np.ascontiguousarray(l)).cuda()).cpu().numpy()
        B0, Bt, Bm, Bg = ev(lam0), ev(lam_tiny), ev(lam_mixed), ev(w.lam)
    assert np.array_equal(B0, Bt)
    assert np.array_equal(Bm[:, 1::2], B0[:, 1::2]) and np.array_equal(Bm[:, ::2], Bg[:, ::2])
    err, _ = vec_relerr(B0, oracle.eval(w, lam=lam0))
    assert err <= TOL_B


def test_eval_linearity_and_shift_invariance(dbie):
    """K-8 symmetries on the GPU path: linear in B0; shifting x0, y0 and the points together."""
    w = workloads.random_boundary(40, 24, seed=11, npts=21)
    B1 = gpu_eval(dbie, w)
    w2 = workloads.random_boundary(40, 24, seed=11, npts=21)
    w2.bx, w2.by, w2.bz = 3.0 * w.bx, -2.0 * w.by, 0.5 * w.bz
    B2 = gpu_eval(dbie, w2)
    assert np.allclose(B2, np.array([3.0, -2.0, 0.5])[:, None] * B1, rtol=1e-13, atol=0)
    w3 = workloads.random_boundary(40, 24, seed=11, npts=21, x0=128.0, y0=-64.0)
    w3.bx, w3.by, w3.bz = w.bx, w.by, w.bz
    w3.x, w3.y, w3.z, w3.lam = w.x + 128.0, w.y - 64.0, w.z, w.lam
    assert np.allclose(gpu_eval(dbie, w3), B1, rtol=1e-11, atol=0)


# ---------------------------------------------------------------------------- eval, fp32 ---
TOL_B_F32 = 2e-4


def _f32_inputs(w):
    """Round the points and lambda to float32 once; the oracle gets exactly those values."""
    w32 = w.subset(np.arange(w.M))
    for k in ("x", "y", "z"):
        setattr(w32, k, getattr(w, k).astype(np.float32).astype(np.float64))
    w32.lam = w.lam.astype(np.float32).astype(np.float64)
    return w32


def gpu_eval_f32(d, w32, mask=0):
    import torch
    with d.DBIE.from_workload(w32, fp32=True) as ctx:
        ctx.set_f32_sfu_mask(mask)
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
        return ctx.eval_f32(t(w32.x), t(w32.y), t(w32.z), t(w32.lam)).cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("mask", [0, 1, 3, 7])
def test_eval_f32_config4_first_points(dbie, mask):
    """BASELINE configs[3], fp32 leg: 512x512 boundary, first 2048 points (4 work blocks of the
    128x4 mapping), every sincos variant; <= 2e-4 relative vector error vs the fp64 oracle."""
    w = _f32_inputs(workloads.config4().subset(np.arange(2048)))
    B = gpu_eval_f32(dbie, w, mask)
    err, dropped = vec_relerr(B, oracle.eval(w))
    assert err <= TOL_B_F32, err
    assert dropped == 0


@pytest.mark.parametrize("nx,ny", [(1, 1), (7, 5), (513, 3), (64, 64), (1030, 2)])
def test_eval_f32_ragged_boundaries(dbie, nx, ny):
    w = _f32_inputs(workloads.random_boundary(nx, ny, seed=nx * 3 + ny, npts=37, h=0.5, x0=-1.0, y0=2.0))
    # the boundary values and pixel centres are rounded to float by dbie_create; use values that
    # are exact in float so that the oracle sees the same boundary
    for k in ("bx", "by", "bz"):
        setattr(w, k, getattr(w, k).astype(np.float32).astype(np.float64))
    err, _ = vec_relerr(gpu_eval_f32(dbie, w), oracle.eval(w), floor=1e-3)
    assert err <= TOL_B_F32, err


def test_eval_f32_host_entry_matches_the_device_entry(dbie):
    """dbie_eval_f32_host (host float arrays, copies inside the call) returns the bits of dbie_eval_f32; it needs the
    fp32 copy of the boundary like the device entry, and M = 0 is a no-op."""
    w = _f32_inputs(workloads.random_boundary(70, 33, seed=8, npts=1111, h=0.5))
    f = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    with dbie.DBIE.from_workload(w, fp32=True) as ctx:
        Bh = ctx.eval_f32_host(f(w.x), f(w.y), f(w.z), f(w.lam))
        assert Bh.dtype == np.float32 and Bh.shape == (3, w.M)
        assert ctx.eval_f32_host(f(w.x[:0]), f(w.y[:0]), f(w.z[:0]), f(w.lam[:, :0])).shape == (3, 0)
    Bd = gpu_eval_f32(dbie, w, mask=7)
    assert np.array_equal(Bh.astype(np.float64), Bd)
    err, _ = vec_relerr(Bd, oracle.eval(w), floor=1e-3)
    assert err <= TOL_B_F32
    with dbie.DBIE.from_workload(w) as ctx:          # no DBIE_WITH_FP32
        with pytest.raises(dbie.DBIEError) as ei:
            ctx.eval_f32_host(f(w.x), f(w.y), f(w.z), f(w.lam))
        assert ei.value.status == dbie.DBIE_ESTATE


def test_eval_f32_needs_the_fp32_copy_and_handles_invalid_points(dbie):
    import torch
    w = _f32_inputs(workloads.random_boundary(20, 12, seed=3, npts=9))
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    with dbie.DBIE.from_workload(w) as ctx:          # no DBIE_WITH_FP32
        with pytest.raises(dbie.DBIEError) as ei:
            ctx.eval_f32(t(w.x), t(w.y), t(w.z), t(w.lam))
        assert ei.value.status == dbie.DBIE_ESTATE
    with dbie.DBIE.from_workload(w, fp32=True) as ctx:
        z = w.z.copy(); z[2] = 0.0
        B = ctx.eval_f32(t(w.x), t(w.y), t(z), t(w.lam)).cpu().numpy()
        assert np.isnan(B[:, 2]).all() and np.isfinite(np.delete(B, 2, axis=1)).all()
        B2 = ctx.eval_f32(t(w.x), t(w.y), t(z), t(w.lam)).cpu().numpy()
        assert np.array_equal(B, B2, equal_nan=True)
        with pytest.raises(TypeError):
            ctx.eval_f32(t(w.x).double(), t(w.y), t(w.z), t(w.lam))


# ---------------------------------------------------------------------------- residual -----
@pytest.mark.parametrize("case", ["random", "config3"])
def test_residual_matches_oracle(dbie, case):
    """A5: Eq. 8, 9, 13, 14 at given lambda triples (one objective evaluation per point)."""
    if case == "random":
        w = workloads.random_boundary(48, 40, seed=5, npts=133, h=0.25)
        lam = w.lam
    else:
        w, _ = workloads.config3().seeded_subset(96)
        lam = np.random.default_rng(9).uniform(0.0, 0.3, (3, w.M)) / w.h
    ro = oracle.residual(w, lam)
    with dbie.DBIE.from_workload(w) as ctx:
        import torch
        dw = dbie.to_device(w)
        r = ctx.residual(dw.x, dw.y, dw.z, torch.from_numpy(lam).cuda())
        r = {k: v.cpu().numpy() for k, v in r.items()}
    err, _ = vec_relerr(r["B"], ro["B"])
    assert err <= TOL_B
    nB = np.linalg.norm(ro["B"], axis=0)
    # J and div are differences of sums over delta = 1e-3 h: rounding noise 1e-13 |B| / delta
    assert np.all(np.abs(r["J"] - ro["J"]) <= 1e-8 * nB / w.h + 1e-300)
    assert np.all(np.abs(r["div"] - ro["div"]) <= 1e-8 * nB / w.h + 1e-300)
    assert np.abs(r["f"] - ro["f"]).max() <= TOL_FG
    assert np.abs(r["g"] - ro["g"]).max() <= TOL_FG
    assert np.abs(r["phi"] - ro["phi"]).max() <= 2 * TOL_FG


@pytest.mark.parametrize("alpha", [0.3, -0.3])
def test_residual_on_the_constant_alpha_packet_gives_J_equal_alpha_B(dbie, alpha):
    """Pin K-12 on the CUDA path: on the constant-alpha force-free packet (workloads/lff.py) at lambda = alpha,
    dbie_residual returns J = alpha B against the closed-form field (not against its own B), div B = 0, f = g = 0
    up to the differences of Eq. 13 / the quadrature of the analytic gradient; J . B has the sign of alpha; at
    lambda = 0 the residuals are two orders larger.  And it agrees with the oracle element by element."""
    import torch
    from workloads.lff import LFFPacket
    w, ref = LFFPacket(alpha).workload()
    nB = np.linalg.norm(ref, axis=0)
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        for analytic, tolJ, tolf, tolg in ((0, 6e-3, 5e-3, 2e-4), (1, 1e-4, 1e-4, 5e-6)):
            lam = np.full((3, w.M), alpha)
            r = ctx.residual(dw.x, dw.y, dw.z, torch.from_numpy(lam).cuda(), dbie.default_opts(analytic=analytic))
            r = {k: v.cpu().numpy() for k, v in r.items()}
            assert (np.linalg.norm(r["B"] - ref, axis=0) / nB).max() <= 1e-5
            dJ = np.linalg.norm(r["J"] - alpha * ref, axis=0) / (abs(alpha) * nB)
            assert dJ.max() <= tolJ, (analytic, dJ.max())
            assert np.all(np.sign((r["J"] * ref).sum(axis=0)) == np.sign(alpha))
            assert (np.abs(r["div"]) * w.h / nB).max() <= 6 * tolg
            assert r["f"].max() <= tolf and r["g"].max() <= tolg
            ro = oracle.residual(w, lam, oracle.Opts(analytic=analytic))
            assert vec_relerr(r["B"], ro["B"])[0] <= TOL_B
            assert np.all(np.abs(r["J"] - ro["J"]) <= 1e-8 * nB / w.h)
            assert np.abs(r["f"] - ro["f"]).max() <= TOL_FG and np.abs(r["g"] - ro["g"]).max() <= TOL_FG
            r0 = ctx.residual(dw.x, dw.y, dw.z, torch.zeros((3, w.M), dtype=torch.float64, device="cuda"),
                              dbie.default_opts(analytic=analytic))
            assert float(r0["f"].min()) >= 0.02 and float(r0["f"].max()) >= 0.2 and float(r0["g"].max()) >= 1e-2


def test_residual_large_delta_takes_the_plain_stencil_path(dbie):
    """MODE_STENCIL4 derives the offset positions from one sincos per component only while lambda*delta <= 1e-3;
    with delta = 0.05 h and lambda up to 0.3/h (lambda*delta = 1.5e-2) most threads take the plain
    four-sincos path, the lambda = 0 points of the same warps the shared-sincos one (divergent warps)."""
    import torch
    w = workloads.random_boundary(48, 40, seed=15, npts=200, h=0.25)
    lam = np.random.default_rng(4).uniform(0.0, 0.3, (3, w.M)) / w.h
    lam[:, ::3] = 0.0
    lam[:, 1::7] *= 0.01
    for delta in (0.05, 1e-3):
        oo = oracle.Opts(delta=delta)
        ro = oracle.residual(w, lam, oo)
        with dbie.DBIE.from_workload(w) as ctx:
            dw = dbie.to_device(w)
            r = ctx.residual(dw.x, dw.y, dw.z, torch.from_numpy(lam).cuda(), dbie.default_opts(delta=delta))
            r = {k: v.cpu().numpy() for k, v in r.items()}
        err, _ = vec_relerr(r["B"], ro["B"])
        assert err <= TOL_B
        nB = np.linalg.norm(ro["B"], axis=0)
        assert np.all(np.abs(r["J"] - ro["J"]) <= 1e-11 * nB / (delta * w.h) + 1e-300)
        assert np.all(np.abs(r["div"] - ro["div"]) <= 1e-11 * nB / (delta * w.h) + 1e-300)
        assert np.abs(r["f"] - ro["f"]).max() <= TOL_FG and np.abs(r["g"] - ro["g"]).max() <= TOL_FG


# ---------------------------------------------------------------------------- solve --------
def _check_solve_parity(dbie, wl, opts_kw=None, gpu=None, min_same=0.99):
    """Protocol P-4; opts_kw["method"] = 1 selects GRID on both sides.
    `gpu`: results already computed on the GPU for exactly the points of `wl` (a sample of a
    larger launch); otherwise the points of `wl` are solved here.

    Every valid point falls in one of two classes, decided from the OUTPUTS only:
      same   : identical status and iteration count AND | |lam|_gpu - |lam|_orc | h <= 1e-6 in all three
               components.  At least `min_same` of the valid points must be in this class (north_star:
               "converged lambda must agree to <= 1e-6").  Where lambda is identical (to 1e-12 / h: the same
               decisions throughout; the simplex vertices are affine combinations of earlier vertices, so
               lambda does not depend on the values of Phi) B must agree to 1e-9 and f, g to 1e-6 directly.
      forked : everything else.  A fork is legitimate only where some comparison of the oracle's search
               was within the noise of a tie (margin < MARGIN_STABLE).
    Every point whose lambda is not identical (forked, or `same` with a late GRID near-tie that moved lambda
    by less than the tolerance) is cross-evaluated: the ORACLE's objective at the GPU's lambda must be as good
    as its own (<= Phi* + 1e-6) and the oracle's B, f, g at the GPU's lambda must match the GPU's."""
    opts_kw = opts_kw or {}
    oo = oracle.Opts(**opts_kw)
    grid = oo.method == 1
    so = oracle.solve_grid(wl, oo) if grid else oracle.solve_nm(wl, oo)
    cnt = None
    if gpu is not None:
        s = gpu
    else:
        with dbie.DBIE.from_workload(wl) as ctx:
            dw = dbie.to_device(wl)
            s = ctx.solve(dw.x, dw.y, dw.z, dbie.default_opts(**opts_kw))
            s = {k: v.cpu().numpy() for k, v in s.items()}
            cnt = ctx.counters()
    valid = so["status"] != 3
    assert np.array_equal(s["status"] == 3, ~valid)
    nvalid = int(valid.sum())
    with np.errstate(invalid="ignore"):
        dlam = np.abs(s["lam"] - so["lam"]).max(axis=0) * wl.h
    same = valid & (s["status"] == so["status"]) & (s["iters"] == so["iters"]) & (dlam <= TOL_LAM)
    forked = valid & ~same
    stable = valid & (so["margin"] >= MARGIN_STABLE)
    info = dict(valid=nvalid, same=int(same.sum()), forked=int(forked.sum()), stable=int(stable.sum()),
                same_frac=float(same.sum()) / max(nvalid, 1),
                max_dlam_h=float(dlam[same].max()) if same.any() else 0.0)
    print(f"P-4 {wl.name}{' ' + str(opts_kw) if opts_kw else ''}: valid {nvalid}, same path and lambda {info['same']} "
          f"({100 * info['same_frac']:.1f} %, max |dlam| h {info['max_dlam_h']:.1e}), forked {info['forked']}, "
          f"oracle margin >= {MARGIN_STABLE:g}: {info['stable']}")
    ident = same & (dlam <= 1e-12)
    if nvalid:
        assert same.any(), "no point of the batch follows the oracle's path"
        # small samples: one fork of a handful of points is allowed
        assert info["same_frac"] >= min(min_same, 1.0 - 1.5 / nvalid), info
    if ident.any():
        err, _ = vec_relerr(s["B"][:, ident], so["B"][:, ident])
        assert err <= TOL_B, err
        assert np.abs(s["f"] - so["f"])[ident].max() <= TOL_FG
        assert np.abs(s["g"] - so["g"])[ident].max() <= TOL_FG
    # a point whose every comparison was clear of the noise must not fork
    assert not (forked & stable).any(), (np.where(forked & stable)[0], so["margin"][forked & stable])
    # lambda not identical: the oracle's own objective at the GPU's lambda is as good, and B, f, g match there
    cross = valid & ~ident
    info["cross"] = int(cross.sum())
    if cross.any():
        sub = wl.subset(np.where(cross)[0])
        ro = oracle.residual(sub, s["lam"][:, cross], oo)
        assert np.all(ro["phi"] <= so["phi"][cross] + 1e-6)
        err, _ = vec_relerr(s["B"][:, cross], ro["B"])
        assert err <= TOL_B
        assert np.abs(s["f"][cross] - ro["f"]).max() <= TOL_FG and np.abs(s["g"][cross] - ro["g"]).max() <= TOL_FG
    # invariants S-2 on the GPU result
    assert np.all(s["lam"][:, valid] >= 0.0)
    st0 = s["status"] == 0
    assert np.all(s["f"][st0] <= oo.eps_f) and np.all(s["g"][st0] <= oo.eps_g)
    if cnt is None:
        pass
    elif grid:   # T candidate values per component per level a point was active in
        assert cnt["objective_evals"] == oo.n_trial * so["iters"][valid].sum() or forked.any()
    else:
        assert cnt["objective_evals"] == so["nfev"][valid].sum() or forked.any()
    return s, so, info


def test_solve_config2_lowlou_subset(dbie):
    """BASELINE configs[1] (Low & Lou n=1, m=1, l=0.3, Phi=pi/4, 64x64 boundary): full NM solve
    on a seeded 160-point subset of the 64x64x32 volume."""
    w, _ = workloads.config2().seeded_subset(160)
    s, so, info = _check_solve_parity(dbie, w)
    # S-3: DBIE's force-free residual is far below the potential field's (lambda = 0)
    pot = oracle.residual(w, np.zeros((3, w.M)))
    assert np.nanmean(s["f"]) < 0.5 * np.nanmean(pot["f"])


def test_solve_config3_bipolar_subset(dbie):
    """BASELINE configs[2] (256x256 at 0.5 Mm/px; h != 1 exercises the units): 40 points."""
    w, _ = workloads.config3().seeded_subset(40)
    _check_solve_parity(dbie, w)


def test_solve_random_boundary_options_and_invalid_points(dbie):
    """Small ragged boundary, non-default options (no Eq. 12 exit, other simplex, low maxiter),
    two invalid points in the batch."""
    w = workloads.random_boundary(33, 21, seed=21, npts=70, h=2.0, zmin=1.5, zmax=6.0)
    w.z[4] = -1.0
    w.x[9] = float("nan")
    s, so, info = _check_solve_parity(dbie, w, dict(use_eq12=0, lam0=0.08, step=0.03, maxiter=37,
                                                    xtol=1e-5, ftol=1e-8, w_g=2.0, cell=0.5))
    assert s["status"][4] == 3 and s["status"][9] == 3
    assert np.isnan(s["lam"][:, 4]).all() and np.isnan(s["B"][:, 9]).all()
    assert (s["status"] == 2).any()      # the iteration cap is reached by some points


def test_solve_and_residual_accept_an_empty_batch(dbie):
    """M = 0 is a valid no-op for every entry point (no launch, empty outputs)."""
    import torch
    w = workloads.random_boundary(20, 12, seed=3, npts=4)
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    with dbie.DBIE.from_workload(w) as ctx:
        for o in (None, dbie.default_opts(method=1), dbie.default_opts(analytic=1)):
            s = ctx.solve(e, e, e, o)
            assert s["B"].shape == (3, 0) and s["status"].numel() == 0
        r = ctx.residual(e, e, e, torch.empty((3, 0), dtype=torch.float64, device="cuda"))
        assert r["J"].shape == (3, 0)
        h = ctx.solve_host(np.empty(0), np.empty(0), np.empty(0))
        assert h["lam"].shape == (3, 0)


def test_solve_is_reproducible_and_host_entry_matches(dbie):
    w, _ = workloads.config2().seeded_subset(64, seed_offset=3)
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        a = ctx.solve(dw.x, dw.y, dw.z)
        b = ctx.solve(dw.x, dw.y, dw.z)
        h = ctx.solve_host(w.x, w.y, w.z)
        for k in ("B", "lam", "f", "g", "iters", "status"):
            assert np.array_equal(a[k].cpu().numpy(), b[k].cpu().numpy(), equal_nan=True), k
            assert np.array_equal(a[k].cpu().numpy(), h[k], equal_nan=True), k
        # J = curl B and div B at the converged lambda (Eq. 14): consistent with the returned f, g
        c = ctx.solve(dw.x, dw.y, dw.z, with_current=True)
        J, B, dv = c["J"].cpu().numpy(), c["B"].cpu().numpy(), c["div"].cpu().numpy()
        nB, nJ = np.linalg.norm(B, axis=0), np.linalg.norm(J, axis=0)
        f = np.linalg.norm(np.cross(J.T, B.T), axis=1) / (nJ * nB)
        assert np.allclose(f, c["f"].cpu().numpy(), atol=1e-7)
        assert np.allclose(np.abs(dv) * (w.h / 6.0) / nB, c["g"].cpu().numpy(), atol=1e-7)
        # maxiter = 0: the best initial vertex is returned with status 2
        z = ctx.solve(dw.x, dw.y, dw.z, dbie.default_opts(maxiter=0))
        assert (z["status"].cpu().numpy() == 2).all() and (z["iters"].cpu().numpy() == 0).all()


# ---------------------------------------------------------------------------- GRID ---------
def test_grid_config2_lowlou_subset(dbie):
    """GRID mode (O-4) with the defaults T = 8, 10 levels on the config-2 boundary."""
    w, _ = workloads.config2().seeded_subset(96, seed_offset=11)
    s, so, info = _check_solve_parity(dbie, w, dict(method=1))
    # after 10 levels the window is 0.4 (2/7)^9 wide: the best two candidates of the last levels
    # differ by less than the 1e-7 margin at about half of the points, which then fall under part
    # (3) of the protocol (cross-evaluation by the oracle) instead of part (2)
    assert info["stable"] >= 0.25 * w.M
    # Phi of the GRID result is not worse than the best of its own level-0 lattice (monotone levels)
    lvl0 = oracle.solve_grid(w, oracle.Opts(method=1, n_level=1, use_eq12=0))
    ok = (s["status"] != 3) & (lvl0["status"] != 3)
    assert np.all((s["f"] + s["g"])[ok] <= lvl0["phi"][ok] + 1e-12)


def test_grid_config5_delta_spot_subset(dbie):
    """BASELINE configs[4]: 1024x1024 boundary (two row segments per row, 2048 tiles, 16 chunks),
    GRID solve with T = 8 on a seeded 12-point subset of the 256x256x128 volume, 4 levels
    (the oracle costs 1.3e8 interactions per point and level)."""
    w, _ = workloads.config5().seeded_subset(12)
    _check_solve_parity(dbie, w, dict(method=1, n_level=4))


@pytest.mark.parametrize("T,levels", [(4, 3), (5, 4), (6, 3), (12, 2)])
def test_grid_trial_counts_options_and_invalid_points(dbie, T, levels):
    """T not a multiple of 8 (4, 2 or 1 trial triples per thread); odd T (the centre trial of every
    refined window coincides with the incumbent, so the level argmin is an exact or near tie at every
    point: whichever of the two wins, lambda is the same to an ulp, so these points still land in the
    `same` class), non-default options, invalid points in the batch, h != 1.  T < 4 is rejected (the
    window 2W/(T-1) would not shrink)."""
    w = workloads.random_boundary(33, 21, seed=50 + T, npts=45, h=2.0, zmin=1.5, zmax=6.0)
    w.z[4] = -1.0
    w.x[9] = float("nan")
    s, so, info = _check_solve_parity(dbie, w, dict(method=1, n_trial=T, n_level=levels, lam_max=0.6,
                                                    use_eq12=0, w_g=2.0, cell=0.5))
    assert s["status"][4] == 3 and s["status"][9] == 3
    valid = so["status"] != 3
    assert np.all(s["iters"][valid] == levels) and np.all(s["status"][valid] == 1)
    assert np.all(s["lam"][:, valid] * w.h <= 0.6 + 1e-12)


def test_grid_is_reproducible_and_host_entry_matches(dbie):
    w, _ = workloads.config2().seeded_subset(50, seed_offset=5)
    o = dbie.default_opts(method=1, n_level=5)
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        a = ctx.solve(dw.x, dw.y, dw.z, o)
        b = ctx.solve(dw.x, dw.y, dw.z, o)
        h = ctx.solve_host(w.x, w.y, w.z, o)
        for k in ("B", "lam", "f", "g", "iters", "status"):
            assert np.array_equal(a[k].cpu().numpy(), b[k].cpu().numpy(), equal_nan=True), k
            assert np.array_equal(a[k].cpu().numpy(), h[k], equal_nan=True), k
        for bad in (dict(n_trial=1), dict(n_trial=2), dict(n_trial=3), dict(n_trial=33), dict(n_level=0),
                    dict(lam_max=0.0)):
            with pytest.raises(dbie.DBIEError):
                ctx.solve(dw.x, dw.y, dw.z, dbie.default_opts(method=1, **bad))


# ------------------------------------------------------------- full-size launches, sampled -
def _solve_full_and_sample(dbie, wl, nsample, opts_kw=None):
    """Solve ALL points of `wl` in one call (the launch configuration bench.py times: persistent
    grid, device-side active lists, many work blocks and a ragged tail) and hand a seeded sample of
    the outputs to the P-4 comparison: points are independent, so a point's result must not depend
    on the batch it was solved in."""
    with dbie.DBIE.from_workload(wl) as ctx:
        dw = dbie.to_device(wl)
        s = ctx.solve(dw.x, dw.y, dw.z, dbie.default_opts(**(opts_kw or {})))
        s = {k: v.cpu().numpy() for k, v in s.items()}
        cnt = ctx.counters()
    npos = 1.0 if (opts_kw or {}).get("analytic") else 4.0     # evaluation positions per objective evaluation
    assert cnt["interactions"] == cnt["objective_evals"] * npos * wl.N
    assert np.isin(s["status"], [0, 1, 2]).all()          # every point of the volume is valid
    assert np.isfinite(s["B"]).all() and (s["lam"] >= 0).all()
    sub, idx = wl.seeded_subset(nsample, seed_offset=77)
    g = {k: (v[:, idx] if v.ndim == 2 else v[idx]) for k, v in s.items()}
    # the same points solved alone (a few dozen points: the warp-per-point shape of the fused kernel, one
    # batch) give the same bits as inside the large launch (thread-per-point shape)
    with dbie.DBIE.from_workload(sub) as ctx:
        dw = dbie.to_device(sub)
        alone = {k: v.cpu().numpy() for k, v in ctx.solve(dw.x, dw.y, dw.z, dbie.default_opts(**(opts_kw or {}))).items()}
    for k in g:
        assert np.array_equal(alone[k], g[k], equal_nan=True), k
    return _check_solve_parity(dbie, sub, opts_kw, gpu=g), s


def test_solve_config2_full_volume_sampled(dbie):
    """BASELINE configs[1] exactly as bench.py runs it: NM solve of all 64x64x32 = 131,072 points;
    96 sampled points are re-solved one by one by the oracle.  S-2/S-3 statistics over the volume."""
    w = workloads.config2()
    (_, so, info), s = _solve_full_and_sample(dbie, w, 96)
    assert info["forked"] <= 2
    # order of magnitude of the paper's residual statistics (<f> 0.078, <g> 6.7e-4)
    assert 0.005 < float(np.mean(s["f"])) < 0.3
    assert float(np.mean(s["g"])) < 0.05


def test_solve_config3_large_batch_sampled(dbie):
    """BASELINE configs[2] boundary (256x256, h = 0.5): NM solve of the 65,536-point seeded subset of
    the 128x128x64 volume that `bench.py --workload cfg3 --points 65536` times (same seed), in one
    call; 24 of them re-solved by the oracle."""
    w, _ = workloads.config3().seeded_subset(65536, seed_offset=900)
    _solve_full_and_sample(dbie, w, 24)


def test_solve_config3_whole_volume_sampled(dbie):
    """BASELINE configs[2] at full size: NM solve of all 128 x 128 x 64 = 1,048,576 points of the 256x256
    boundary in ONE dbie_solve call (about 3 minutes of FP64 work); 64 sampled points are re-solved by the
    oracle, and solved again alone on the GPU (bit-identical)."""
    w = workloads.config3()
    assert w.M == 1048576
    (_, _, info), s = _solve_full_and_sample(dbie, w, 64)
    assert info["forked"] <= 1
    assert 0.005 < float(np.mean(s["f"])) < 0.5


def test_grid_config5_ten_levels_as_benched(dbie):
    """BASELINE configs[4] with exactly the options bench.py times (GRID, T = 8, 10 levels) on the
    1024x1024 boundary: 16 seeded points against orc_solve_grid, Eq. 13 differences and the analytic
    gradient.  After ten levels the window is 0.4 (2/7)^9 = 5e-6 wide, so late near-ties move lambda by
    less than the 1e-6 tolerance; a fork at an early level would not."""
    w, _ = workloads.config5().seeded_subset(16, seed_offset=31)
    for kw in (dict(method=1), dict(method=1, analytic=1)):
        s, so, info = _check_solve_parity(dbie, w, kw)
        assert np.all(so["iters"][so["status"] == 1] == 10)


def test_grid_config5_large_batch_sampled(dbie):
    """BASELINE configs[4] boundary (1024x1024): GRID solve (T = 8; 3 of the 10 levels, the oracle
    costs 1.3e8 interactions per point and level) of the 16,384-point seeded subset of the
    256x256x128 volume that `bench.py --workload cfg5` times (same seed), in one call; 6 of them
    re-solved by the oracle."""
    w, _ = workloads.config5().seeded_subset(16384, seed_offset=900)
    _solve_full_and_sample(dbie, w, 6, dict(method=1, n_level=3))


def test_grid_config5_z_slab_at_the_timed_shape(dbie):
    """BASELINE configs[4] at the launch shape `bench.py --slabs` times and projects the full volume from: ONE
    z-slab of 256 x 256 = 65,536 points (z = 32 px) of the 256x256x128 volume, 1024x1024 boundary, GRID with
    T = 8 and all 10 levels, in one dbie_solve call.  8 seeded points of the slab are re-solved by
    orc_solve_grid (2.7e9 oracle interactions) and solved again alone on the GPU (bit-identical)."""
    full = workloads.config5()
    per = full.M // 128
    assert per == 65536
    slab = full.subset(np.arange(31 * per, 32 * per))
    assert np.all(slab.z == slab.z[0]) and abs(slab.z[0] / full.h - 32.0) < 1e-9
    (_, so, info), s = _solve_full_and_sample(dbie, slab, 8, dict(method=1))
    assert np.all(so["iters"][so["status"] == 1] == 10)
    assert np.isin(s["iters"], np.arange(1, 11)).all()


def test_eval_f32_config4_full_size_sampled(dbie):
    """BASELINE configs[3], fp32 leg, in the launch configuration bench.py times: the full M = 1,048,576 launch
    of dbie_eval_f32 (unsplit work items, fp64 chunk sums); 192 seeded outputs recomputed one by one by the fp64
    oracle (<= 2e-4 relative vector error), and the launch is bitwise reproducible."""
    import torch
    w = _f32_inputs(workloads.config4())
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    with dbie.DBIE.from_workload(w, fp32=True) as ctx:
        x, y, z, lam = t(w.x), t(w.y), t(w.z), t(w.lam)
        B = ctx.eval_f32(x, y, z, lam)
        B2 = ctx.eval_f32(x, y, z, lam)
        assert torch.equal(B, B2) and bool(torch.isfinite(B).all())
        assert ctx.counters()["interactions"] == float(w.M) * w.N
        # a result does not depend on the batch it was computed in (chunk sums in canonical order)
        idx = torch.arange(70000, 70000 + 1500, device="cuda")
        Bs = ctx.eval_f32(x[idx].contiguous(), y[idx].contiguous(), z[idx].contiguous(), lam[:, idx].contiguous())
        assert torch.equal(Bs, B[:, idx])
        B = B.cpu().numpy().astype(np.float64)
    sub, idx = w.seeded_subset(192)
    err, dropped = vec_relerr(B[:, idx], oracle.eval(sub))
    assert err <= TOL_B_F32 and dropped == 0, err


# ------------------------------------------- analytic gradient (O-5) -
@pytest.mark.parametrize("case", ["random", "config3", "config5"])
def test_analytic_residual_matches_oracle(dbie, case):
    """dbie_residual with opts.analytic = 1 against orc_residual(analytic = 1): B to 1e-9; J and
    div B are direct sums now (no division by delta), so they match to 1e-9 of |grad B| as well."""
    import torch
    if case == "random":
        w = workloads.random_boundary(37, 23, seed=12, npts=300, h=0.5, x0=-3.0, y0=1.0, zmin=0.6, zmax=8.0)
        lam = w.lam
    elif case == "config3":
        w, _ = workloads.config3().seeded_subset(96)
        lam = np.random.default_rng(9).uniform(0.0, 0.3, (3, w.M)) / w.h
    else:
        w, _ = workloads.config5().seeded_subset(24)
        lam = np.random.default_rng(10).uniform(0.0, 0.3, (3, w.M)) / w.h
    oo = oracle.Opts(analytic=1)
    ro = oracle.residual(w, lam, oo)
    _, G = oracle.gradient(w, lam)
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        r = ctx.residual(dw.x, dw.y, dw.z, torch.from_numpy(np.ascontiguousarray(lam)).cuda(),
                         dbie.default_opts(analytic=1))
        r = {k: v.cpu().numpy() for k, v in r.items()}
        assert ctx.counters()["interactions"] == float(w.M) * w.N
    err, _ = vec_relerr(r["B"], ro["B"])
    assert err <= TOL_B
    gscale = np.abs(G).max(axis=(0, 1))
    assert np.all(np.abs(r["J"] - ro["J"]) <= 1e-9 * gscale)
    assert np.all(np.abs(r["div"] - ro["div"]) <= 1e-9 * gscale)
    assert np.abs(r["f"] - ro["f"]).max() <= TOL_FG
    assert np.abs(r["g"] - ro["g"]).max() <= TOL_FG
    assert np.abs(r["phi"] - ro["phi"]).max() <= 2 * TOL_FG


def test_analytic_solve_config2_subset_and_full_volume(dbie):
    """NM solve with the analytic gradient: P-4 parity on a 160-point subset of config 2, then the
    whole 131,072-point volume in one call with 64 sampled points re-solved by the oracle."""
    w, _ = workloads.config2().seeded_subset(160)
    s, so, info = _check_solve_parity(dbie, w, dict(analytic=1))
    assert info["forked"] <= 1          # derivative noise ~1e-13: far fewer near-ties than with Eq. 13
    (_, _, info2), sfull = _solve_full_and_sample(dbie, workloads.config2(), 64, dict(analytic=1))
    assert 0.005 < float(np.mean(sfull["f"])) < 0.3


def test_analytic_solve_config3_options_and_invalid_points(dbie):
    w, _ = workloads.config3().seeded_subset(32, seed_offset=2)
    w.z[3] = 0.0
    s, so, info = _check_solve_parity(dbie, w, dict(analytic=1, use_eq12=0, maxiter=60, w_g=2.0, cell=0.5))
    assert s["status"][3] == 3


@pytest.mark.parametrize("T,levels", [(8, 6), (5, 3)])
def test_analytic_grid_config2_subset(dbie, T, levels):
    """GRID search on the analytic gradient (O-4 + O-5): even and odd T."""
    w, _ = workloads.config2().seeded_subset(64, seed_offset=13)
    _check_solve_parity(dbie, w, dict(method=1, analytic=1, n_trial=T, n_level=levels))


def test_analytic_grid_config5_large_batch_sampled(dbie):
    """BASELINE configs[4] boundary: GRID (T = 8, 3 levels) with the analytic gradient on a
    4,096-point subset in one call; 6 sampled points re-solved by the oracle."""
    w, _ = workloads.config5().seeded_subset(4096, seed_offset=6)
    _solve_full_and_sample(dbie, w, 6, dict(method=1, analytic=1, n_level=3))


def test_fp64_operand_probe_shows_the_three_register_penalty(dbie):
    """dbie_probe_fp64_operands (the measurement behind DESIGN.md section 6): two-register FP64 instructions run at
    the FP64 pipe's rate, a DFMA reading three different registers at about two thirds of it."""
    r = dbie.probe_fp64_operands(30.0)
    peak = 148 * 64 * 1.965e9
    assert 0.5 * peak < r["dfma_2reg_imm"] < 1.05 * peak           # loose: the SM clock is the box's business
    assert abs(r["dmul"] / r["dfma_2reg_imm"] - 1.0) < 0.05
    assert 0.55 * r["dfma_2reg_imm"] < r["dfma_3reg"] < 0.8 * r["dfma_2reg_imm"]
    assert r["dfma_3reg"] < r["dfma_1reg_2reuse"] <= 1.02 * r["dfma_2reg_imm"]


# ---------------------------------------------- the paper's own validation case --
PAPER_TABLE1 = {   # PAPER.md:145-159, Table 1 (printed values)
    "paper: Present DBIE Method": (0.99, 0.52, 0.83, -0.53, 1.08),
    "paper: Boundary Integral Method (no iteration)": (0.97, 0.41, -0.02, -14.0, 1.00),
}


def test_lowlou_case2_figures_of_merit(dbie, capsys):
    """PAPER.md:145-163 / Table 1: Low & Lou n = 3, m = 1, l = 0.3, Phi = 4 pi/5, 192x192 boundary around the 64^3
    region, "bottom boundary only".  Gated: the pipeline runs at the paper's size, the GPU results match the oracle
    on sampled points (P-4), and the solved field is far more force-free than the potential field.  NOT gated: the
    five figures of merit.  Table 1's "Present DBIE" row is not reproduced under the readings of DESIGN.md section 3
    (parity unpinned); the table printed here (pytest -s) records what each open reading gives,
    next to the paper's two rows, without freezing this build's own numbers into a test."""
    import dataclasses
    import torch
    w = workloads.lowlou_case2()
    ll, scale = w.extra["lowlou"], w.extra["scale"]
    exact = lambda wl: np.array(ll.field(wl.x, wl.y, wl.z)) * scale
    rows = {}

    def fom(name, wl, B):
        m = workloads.figures_of_merit(exact(wl), B)
        rows[name] = (m["C_vec"], m["C_cs"], m["E_n_prime"], m["E_m_prime"], m["eps"])

    def gpu_eval_at(wl, lam):
        with dbie.DBIE.from_workload(wl) as ctx:
            dw = dbie.to_device(wl)
            return ctx.eval(dw.x, dw.y, dw.z, torch.from_numpy(np.ascontiguousarray(lam)).cuda()).cpu().numpy()

    def gpu_solve(wl, **kw):
        with dbie.DBIE.from_workload(wl) as ctx:
            dw = dbie.to_device(wl)
            return {k: v.cpu().numpy() for k, v in ctx.solve(dw.x, dw.y, dw.z, dbie.default_opts(**kw)).items()}

    # the gated part: one full-volume solve, sampled against the oracle
    (_, _, info), s = _solve_full_and_sample(dbie, w, 24, dict(analytic=1))
    fom("NM solve, defaults (analytic gradient)", w, s["B"])
    pot = gpu_eval_at(w, np.zeros((3, w.M)))
    fom("lambda = 0 (potential field of the window)", w, pot)
    pot_res = None
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        pot_res = ctx.residual(dw.x, dw.y, dw.z, torch.zeros((3, w.M), dtype=torch.float64, device="cuda"),
                               dbie.default_opts(analytic=1))["f"].cpu().numpy()
    assert float(np.mean(s["f"])) < 0.5 * float(np.nanmean(pot_res))    # far more force-free than the potential field
    assert float(np.mean(s["f"])) < 0.2

    # the reported part: open readings, one at a time
    al = np.abs(ll.alpha(w.x, w.y, w.z))
    fom("lambda = the exact alpha of the model field, all three components", w, gpu_eval_at(w, np.tile(al, (3, 1))))
    fom("NM solve, Eq. 13 finite differences", w, gpu_solve(w)["B"])
    fom("NM solve, Phi = f only (w_g = 0)", w, gpu_solve(w, analytic=1, w_g=0.0)["B"])
    fom("NM solve, Phi = f + 10 g", w, gpu_solve(w, analytic=1, w_g=10.0)["B"])
    fom("NM solve, start and step 0.5 / h", w, gpu_solve(w, analytic=1, lam0=0.5, step=0.5)["B"])
    w_half = dataclasses.replace(w, z=w.z - 0.5 * w.h)
    fom("NM solve, layers at z = (k + 1/2) h", w_half, gpu_solve(w_half, analytic=1)["B"])
    w9 = dataclasses.replace(w, quad=9)
    fom("NM solve, 9-node element quadrature (O-6)", w9, gpu_solve(w9, analytic=1)["B"])
    fom("NM solve, start 0.15 / h, step 0.05 / h", w, gpu_solve(w, analytic=1, lam0=0.15, step=0.05)["B"])
    # the same window with its outer 32 pixels tapered to zero (the paper asks for a boundary that
    # "approaches zero" at the edge), to separate the truncation of the window from the method
    ramp = np.clip((np.arange(w.nx) + 0.5) / 32.0, 0.0, 1.0)
    t1 = 0.5 - 0.5 * np.cos(np.pi * np.minimum(ramp, ramp[::-1]))
    taper = np.outer(t1, t1).ravel()
    w_ap = dataclasses.replace(w, bx=w.bx * taper, by=w.by * taper, bz=w.bz * taper)
    fom("lambda = 0, window tapered to zero over its outer 32 pixels", w_ap, gpu_eval_at(w_ap, np.zeros((3, w.M))))
    fom("NM solve, window tapered to zero over its outer 32 pixels", w_ap, gpu_solve(w_ap, analytic=1)["B"])
    # an upper bound for ANY search: per point and component the lambda of a 96-value scan of [0, 0.8 / h] whose
    # B_p is closest to the exact field (uses the answer; not a reconstruction), and the objective there
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        ex = torch.from_numpy(exact(w)).cuda()
        be = torch.full((3, w.M), float("inf"), dtype=torch.float64, device="cuda")
        bl, bB = torch.zeros_like(be), torch.zeros_like(be)
        for lv in np.linspace(0.0, 0.8, 96) / w.h:
            Bl = ctx.eval(dw.x, dw.y, dw.z, torch.full((3, w.M), float(lv), dtype=torch.float64, device="cuda"))
            upd = (Bl - ex).abs() < be
            be = torch.where(upd, (Bl - ex).abs(), be)
            bl = torch.where(upd, torch.full_like(bl, float(lv)), bl)
            bB = torch.where(upd, Bl, bB)
        fom("closest-to-exact lambda per component (96-value scan; uses the answer)", w, bB.cpu().numpy())
        o = dbie.default_opts(analytic=1)
        ri = ctx.residual(dw.x, dw.y, dw.z, bl, o)
        rs = ctx.residual(dw.x, dw.y, dw.z, torch.from_numpy(s["lam"]).cuda(), o)
        phi_note = ("objective at the closest-to-exact lambda: mean f %.3f, mean g %.3f; at the NM solution: mean f %.3f, "
                    "mean g %.4f; Phi(closest-to-exact) < Phi(NM) at %.1f %% of the points"
                    % (float(ri["f"].nanmean()), float(ri["g"].nanmean()), float(rs["f"].nanmean()),
                       float(rs["g"].nanmean()), 100.0 * float((ri["phi"] < rs["phi"]).double().mean())))
    low = w.z <= 16.5 * w.h
    m = workloads.figures_of_merit(exact(w)[:, low], s["B"][:, low])
    rows["NM solve, defaults: metrics over the 16 lowest layers only"] = (m["C_vec"], m["C_cs"], m["E_n_prime"],
                                                                         m["E_m_prime"], m["eps"])
    with capsys.disabled():
        print("\nLow & Lou Case II, figures of merit over the 64^3 region (C_vec, C_cs, E'_n, E'_m, eps):")
        for name, v in list(PAPER_TABLE1.items()) + list(rows.items()):
            print(f"  {name:74s} " + " ".join(f"{x:8.3f}" for x in v))
        print("  " + phi_note)
    for v in rows.values():
        assert all(np.isfinite(v))


# ------------------------------------ 9-node element quadrature (O-6) -
def _q9(w):
    import copy
    w9 = copy.copy(w)
    w9.quad = 9
    return w9


@pytest.mark.parametrize("nx,ny", [(3, 3), (4, 3), (7, 5), (6, 9), (33, 21), (64, 64), (343, 5), (700, 4)])
def test_q9_eval_matches_oracle(dbie, nx, ny):
    """DBIE_QUAD_9NODE: odd / even node counts (half elements), the smallest grid, source rows longer
    than one 512-record tile (343 nodes -> 513 sources; 700 -> 1050), h != 1, shifted origin."""
    w = _q9(workloads.random_boundary(nx, ny, seed=nx * 5 + ny, npts=41, h=0.5, x0=-1.0, y0=2.0))
    w.lam[:, 0] = 0.0
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        B = ctx.eval(dw.x, dw.y, dw.z, dw.lam).cpu().numpy()
        assert ctx.counters()["interactions"] == float(w.M) * (3 * (nx // 2)) * (3 * (ny // 2))
    err, _ = vec_relerr(B, oracle.eval(w))
    assert err <= TOL_B
    # and it is a different discretisation from the one-source-per-pixel rule
    assert not np.allclose(B, gpu_eval(dbie, workloads.random_boundary(nx, ny, seed=nx * 5 + ny, npts=41, h=0.5,
                                                                       x0=-1.0, y0=2.0)), rtol=1e-6)


def test_q9_solve_and_residual_config2(dbie):
    """The whole path on the 9-node sources: Eq. 13 residual, NM solve (Eq. 13 and analytic), GRID."""
    import torch
    w = _q9(workloads.config2().seeded_subset(64, seed_offset=21)[0])
    lam = np.random.default_rng(3).uniform(0.0, 0.3, (3, w.M)) / w.h
    ro = oracle.residual(w, lam)
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        r = {k: v.cpu().numpy() for k, v in ctx.residual(dw.x, dw.y, dw.z, torch.from_numpy(lam).cuda()).items()}
    err, _ = vec_relerr(r["B"], ro["B"])
    assert err <= TOL_B and np.abs(r["f"] - ro["f"]).max() <= TOL_FG and np.abs(r["g"] - ro["g"]).max() <= TOL_FG
    _check_solve_parity(dbie, w)
    _check_solve_parity(dbie, w, dict(analytic=1))
    _check_solve_parity(dbie, w, dict(method=1, n_level=4))


def test_q9_eval_f32_and_bad_sizes(dbie):
    import torch
    w = _q9(_f32_inputs(workloads.random_boundary(65, 40, seed=77, npts=300, zmin=1.0, zmax=30.0)))
    with dbie.DBIE.from_workload(w, fp32=True) as ctx:
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
        B = ctx.eval_f32(t(w.x), t(w.y), t(w.z), t(w.lam)).cpu().numpy().astype(np.float64)
    err, _ = vec_relerr(B, oracle.eval(w))
    assert err <= TOL_B_F32
    with pytest.raises(dbie.DBIEError):
        dbie.DBIE(2, 5, 1.0, 0.0, 0.0, np.ones(10), np.ones(10), np.ones(10), quad9=True)


# ------------------------------------------------ internal batching (dbie_debug_set_batch_limit) -
def test_internal_batches_do_not_change_a_bit(dbie):
    """eval, eval_f32, residual, the Nelder-Mead solve and GRID process large M in internal batches
    (2^21 / 2^22 points, a 2 GiB scratch bound): never reached by the other tests.  With the test knob
    the same paths run with 3-4 uneven batches (offsets > 0, a ragged last batch) and must reproduce the
    single-batch results bit for bit, for every output array."""
    import torch
    w, _ = workloads.config2().seeded_subset(700, seed_offset=4)
    lam = np.random.default_rng(2).uniform(0.0, 0.3, (3, w.M)) / w.h
    w.z[11] = -1.0                                   # an invalid point in the second batch
    t64 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()
    t32 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()

    def run_all(ctx):
        dw = dbie.to_device(w)
        out = {"eval": ctx.eval(dw.x, dw.y, dw.z, t64(lam)),
               "f32": ctx.eval_f32(t32(w.x), t32(w.y), t32(w.z), t32(lam))}
        for name, o in (("res", None), ("res_an", dbie.default_opts(analytic=1))):
            for k, v in ctx.residual(dw.x, dw.y, dw.z, t64(lam), o).items():
                out[f"{name}.{k}"] = v
        for name, o in (("nm", dbie.default_opts(maxiter=40)), ("nm_an", dbie.default_opts(maxiter=40, analytic=1)),
                        ("grid", dbie.default_opts(method=1, n_level=3)),
                        ("grid_an", dbie.default_opts(method=1, n_level=3, analytic=1, n_trial=6))):
            for k, v in ctx.solve(dw.x, dw.y, dw.z, o).items():
                out[f"{name}.{k}"] = v
        return {k: v.cpu().numpy() for k, v in out.items()}

    with dbie.DBIE.from_workload(w, fp32=True) as ctx:
        one = run_all(ctx)
        for limit in (256, 199):                     # 3 batches (256, 256, 188) and 4 (199, 199, 199, 103)
            ctx.set_batch_limit(limit)
            many = run_all(ctx)
            for k in one:
                assert np.array_equal(one[k], many[k], equal_nan=True), (limit, k)
        ctx.set_batch_limit(0)
    assert one["nm.status"][11] == 3 and np.isnan(one["eval"][:, 11]).all()


# ------------------------------------------------------------- range of theta (include/dbie.h) --
@pytest.mark.parametrize("theta", [1e3, 1e4, 1e5])
def test_eval_large_theta_against_oracle(dbie, theta):
    """include/dbie.h: theta = |lambda| r < 2^20.  The kernel's one-step Cody-Waite reduction leaves
    k (pi/128 - fl(pi/128)) = 3.9e-17 theta, and theta = lambda r itself carries half an ulp (1.1e-16 theta) on
    both sides, r possibly one more: each term n(theta) w b is then off by about |theta| * ulp(theta), i.e.
    2^-52 theta relative to its own amplitude.  Gate: |dB| <= 8 * 2^-52 * theta_max * sum |terms|."""
    w = workloads.random_boundary(40, 24, seed=77, npts=64, zmin=2.0, zmax=9.0)
    lam = np.full((3, w.M), 1.0)
    xk = w.x0 + (np.arange(w.nx) + 0.5) * w.h
    yk = w.y0 + (np.arange(w.ny) + 0.5) * w.h
    r = np.sqrt((xk[None, None, :] - w.x[:, None, None]) ** 2 + (yk[None, :, None] - w.y[:, None, None]) ** 2
                + w.z[:, None, None] ** 2)
    lam *= theta / r.max(axis=(1, 2))                         # theta_max = theta at every point
    lam[1] *= 0.37; lam[2] *= 0.81
    with dbie.DBIE.from_workload(w) as ctx:
        import torch
        dw = dbie.to_device(w)
        B = ctx.eval(dw.x, dw.y, dw.z, torch.from_numpy(lam).cuda()).cpu().numpy()
    R = oracle.eval(w, lam=lam)
    c = w.z * w.h ** 2 / (2 * np.pi)
    for p, b0 in enumerate((w.bx, w.by, w.bz)):
        th = lam[p][:, None, None] * r
        mag = c * np.sum((th + 1.0) / r ** 3 * np.abs(b0.reshape(w.ny, w.nx))[None], axis=(1, 2))
        assert np.all(np.abs(B[p] - R[p]) <= 8 * 2.0 ** -52 * theta * mag), (p, np.abs(B[p] - R[p]).max(), mag.min())


# ---------------------------------------- field-line / current-line tracing -----
def _gpu_trace(dbie, w, seeds, topts_kw, sopts_kw=None):
    import torch
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()
    with dbie.DBIE.from_workload(w) as ctx:
        out = ctx.trace(t(seeds[0]), t(seeds[1]), t(seeds[2]), dbie.default_trace_opts(**topts_kw),
                        dbie.default_opts(**(sopts_kw or {})))
        return {k: v.cpu().numpy() for k, v in out.items()}


def _check_trace(g, o, h, tol=1e-8):
    path, npts, status = o
    assert np.array_equal(g["npts"], npts), (g["npts"], npts)
    assert np.array_equal(g["status"], status)
    assert np.array_equal(np.isnan(g["path"]), np.isnan(path))
    d = np.nanmax(np.abs(g["path"] - path)) if np.isfinite(path).any() else 0.0
    assert d <= tol * h, d / h
    return d / h


def test_trace_potential_field_lines_of_the_dipole(dbie):
    """lambda = 0 (fixed): lines of the DBIE field of the buried dipole's magnetogram, GPU against the tracing
    oracle point by point, both directions, with lines that leave through z_min, through the window side and
    seeds outside the region; the GPU lines keep the dipole invariant r / sin^2(theta) like the oracle's (T-4)."""
    from oracle import trace as otrace
    w = workloads.config1(n=64)
    seeds = np.array([[9.5, 8.0, 6.0], [8.0, 6.0, 6.5], [10.0, 10.0, 6.0], [8.0 + 31.0, 8.0, 3.0], [8.0, 8.0 - 31.5, 3.0],
                      [200.0, 8.0, 3.0], [9.0, 9.0, 2.4]]).T.copy()
    for direction in (1, -1):
        kw = dict(ds=0.25, max_steps=50, direction=direction, z_min=2.5)
        g = _gpu_trace(dbie, w, seeds, dict(kw, lam=(0.0, 0.0, 0.0)))
        o = otrace.trace_dbie(w, seeds, otrace.TraceOpts(fixed_lam=(0.0, 0.0, 0.0), **kw))
        _check_trace(g, o, w.h)
        assert list(g["npts"][-2:]) == [0, 0] and (g["status"][-2:] == 1).all()
    p = g["path"][:, :g["npts"][0], 0]
    X, Y, Z = p[0] - 8.0, p[1] - 8.0, p[2] + 4.0
    R = np.sqrt(X * X + Y * Y + Z * Z)
    Lsh = R ** 3 / (X * X + Y * Y)
    assert np.abs(Lsh / Lsh[0] - 1.0).max() < 5e-3       # 64x64 window: truncation 1.4e-3 (pin K-6)


@pytest.mark.parametrize("current", [0, 1])
def test_trace_with_the_lambda_solve_matches_the_oracle(dbie, current):
    """Lines of B (and current lines of J, Eq. 14) with lambda from the per-point Nelder-Mead search at every
    stage point, on the Low & Lou boundary of BASELINE configs[1]: 12 seeds x 6 steps = 288 point solves per
    line set, compared point by point with the oracle's sequential RK4 (1e-8 h).  The search runs in the
    warp-per-point shape of the fused kernel (12 points)."""
    from oracle import trace as otrace
    w, _ = workloads.config2().seeded_subset(12, seed_offset=5)
    seeds = np.stack([w.x, w.y, w.z + 3 * w.h])
    kw = dict(ds=0.5, max_steps=6, direction=1, current=current)
    g = _gpu_trace(dbie, w, seeds, kw)
    o = otrace.trace_dbie(w, seeds, otrace.TraceOpts(**kw))
    d = _check_trace(g, o, w.h)
    print(f"trace current={current}: max |dr| = {d:.1e} h over {int(g['npts'].sum())} points")
    assert g["npts"].max() >= 4


def test_trace_analytic_gradient_and_options(dbie):
    """The analytic-gradient search (O-5) under the tracer, against the field, with a z_max lid, on the config-3
    boundary (h = 0.5); bad options are rejected."""
    import torch
    from oracle import trace as otrace
    w, _ = workloads.config3().seeded_subset(8, seed_offset=8)
    seeds = np.stack([w.x, w.y, np.minimum(w.z, 6.0 * w.h)])
    kw = dict(ds=0.4, max_steps=4, direction=-1, z_min=0.5, z_max=7.0)
    g = _gpu_trace(dbie, w, seeds, kw, dict(analytic=1))
    o = otrace.trace_dbie(w, seeds, otrace.TraceOpts(**kw), oracle.Opts(analytic=1))
    _check_trace(g, o, w.h)
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    with dbie.DBIE.from_workload(w) as ctx:
        out = ctx.trace(e, e, e)
        assert out["path"].shape == (3, 101, 0)
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        for bad in (dict(ds=0.0), dict(direction=0), dict(max_steps=-1), dict(z_min=2.0, z_max=1.0)):
            with pytest.raises(dbie.DBIEError):
                ctx.trace(t(seeds[0]), t(seeds[1]), t(seeds[2]), dbie.default_trace_opts(**bad))


def test_pass_trace_of_the_fused_solve(dbie):
    """dbie_last_pass_trace (profile mode): one entry per pass of the fused Nelder-Mead launch; the active counts
    start at M, never grow, and their sum is the number of objective evaluations the counters report."""
    w, _ = workloads.config2().seeded_subset(3000, seed_offset=5)
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        assert ctx.pass_trace()["npass"] == 0                  # nothing recorded without profile mode
        ctx.solve(dw.x, dw.y, dw.z)
        assert ctx.pass_trace()["npass"] == 0
        ctx.profile(True)
        s = ctx.solve(dw.x, dw.y, dw.z)
        t = ctx.pass_trace()
        c = ctx.counters()
        # the timeline belongs to the LAST call only: an unprofiled solve, a GRID solve, an eval or a residual after
        # the profiled solve invalidates it (it used to keep reporting the old launch)
        import torch
        lam0 = torch.zeros((3, w.M), dtype=torch.float64, device="cuda")
        for other in (lambda: ctx.eval(dw.x, dw.y, dw.z, lam0), lambda: ctx.residual(dw.x, dw.y, dw.z, lam0),
                      lambda: ctx.solve(dw.x[:64].contiguous(), dw.y[:64].contiguous(), dw.z[:64].contiguous(),
                                        dbie.default_opts(method=1, n_level=2))):
            ctx.solve(dw.x, dw.y, dw.z)
            assert ctx.pass_trace()["npass"] == t["npass"]
            other()
            assert ctx.pass_trace()["npass"] == 0
        ctx.profile(False)
        ctx.solve(dw.x, dw.y, dw.z)
        assert ctx.pass_trace()["npass"] == 0
    assert t["npass"] == len(t["active"]) > 50
    assert t["active"][0] == w.M and np.all(np.diff(t["active"]) <= 0) and t["active"][-1] > 0
    assert int(t["active"].sum()) == c["objective_evals"]
    assert np.all(t["ms"] > 0) and t["ms"].sum() < 1e4


def test_maxiter_is_bounded_and_a_capped_search_reports_status_2(dbie):
    """dbie_solve_opts.maxiter above 2^24 is refused (5 maxiter + 5 passes would overflow int near 4.3e8 and the
    fused kernel would then run zero passes and return DBIE_OK with nothing written); maxiter = 0 and 1 are legal
    and every valid point then ends with status 2 (or an earlier stop) and finite outputs."""
    w, _ = workloads.config2().seeded_subset(64, seed_offset=11)
    with dbie.DBIE.from_workload(w) as ctx:
        dw = dbie.to_device(w)
        for bad in ((1 << 24) + 1, 500_000_000, 2 ** 31 - 1, -1):
            with pytest.raises(dbie.DBIEError) as ei:
                ctx.solve(dw.x, dw.y, dw.z, dbie.default_opts(maxiter=bad))
            assert ei.value.status == dbie.DBIE_EINVAL
        ctx.profile(True)                                       # the pass-trace buffer is capped too, not sized from maxiter
        big = ctx.solve(dw.x, dw.y, dw.z, dbie.default_opts(maxiter=1 << 24))
        ref = ctx.solve(dw.x, dw.y, dw.z)
        import torch
        npass_ref = ctx.pass_trace()["npass"]
        m = ref["status"] != 2                                  # points the default cap of 200 did not cut short
        assert int(m.sum()) > 0 and torch.equal(big["lam"][:, m], ref["lam"][:, m]) and torch.equal(big["B"][:, m], ref["B"][:, m])
        assert int((big["status"] == 2).sum()) == 0 and 0 < npass_ref <= 65536
        for mi in (0, 1):
            s = ctx.solve(dw.x, dw.y, dw.z, dbie.default_opts(maxiter=mi))
            st = s["status"].cpu().numpy()
            assert np.all((st == 2) | (st == 0) | (st == 1)) and (st == 2).sum() > 0
            assert bool(torch.isfinite(s["B"]).all()) and int(s["iters"].max()) <= mi
