"""A short program that drives every kernel of libdbie_b200.so once, for compute-sanitizer:

    compute-sanitizer --tool memcheck|racecheck|initcheck python tests/sanitizer_target.py

It is test infrastructure (not collected by pytest: no test_ prefix) and checks nothing against the oracle; it only
has to run every code path at sizes a sanitizer finishes in a minute or two, and print what it ran:
  - dbie_create (nodal and 9-node staging, fp32 copy), dbie_eval (split and unsplit launches), dbie_eval_noalloc,
    dbie_eval_f32, dbie_residual (Eq. 13 stencil and analytic gradient);
  - the fused Nelder-Mead kernel in BOTH of its shapes: 1,500 points of config 2 start thread-per-point with the
    chunk range split over CTAs (the "last arriver adds the partial sums" path and its self-resetting counters) and
    finish warp-per-point once fewer than ~800 points are active; 48 points run warp-per-point throughout;
    two internal batches exercise the counter reset between launches;
  - one GRID solve (T = 8, 3 levels) and one on the analytic gradient (T = 4);
  - a 2-seed field-line trace with the lambda search at every stage point and a current-line trace at fixed lambda.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    import torch
    import workloads
    import paper_1306_1122_b200 as dbie

    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    dbie.load()
    ran = []
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()

    # eval paths on a ragged boundary (rows shared between chunks), 9-node staging, fp32
    w = workloads.random_boundary(96, 80, seed=1, npts=700, h=0.7, x0=-3.0, y0=1.5)
    d = dbie.to_device(w)
    with dbie.DBIE.from_workload(w, fp32=True) as ctx:
        B = ctx.eval(d.x, d.y, d.z, d.lam)
        out = torch.empty_like(B)
        ctx.eval_noalloc(d.x, d.y, d.z, d.lam, out)
        assert torch.equal(B, out)
        ctx.eval_f32(d.x.float(), d.y.float(), d.z.float(), d.lam.float())
        ctx.residual(d.x, d.y, d.z, d.lam)
        ctx.residual(d.x, d.y, d.z, d.lam, dbie.default_opts(analytic=1))
        ctx.set_batch_limit(300)                       # three internal batches, a ragged last one
        assert torch.equal(ctx.eval(d.x, d.y, d.z, d.lam), B)
        ran.append("eval/noalloc/f32/residual 96x80 x 700")
    with dbie.DBIE(w.nx, w.ny, w.h, w.x0, w.y0, w.bx, w.by, w.bz, quad9=True) as ctx:
        ctx.eval(d.x, d.y, d.z, d.lam)
        ran.append("9-node eval")
    wide = workloads.random_boundary(1030, 3, seed=2, npts=300000 // 1030, h=0.5)   # row segments (nx > 512)
    dw = dbie.to_device(wide)
    with dbie.DBIE.from_workload(wide) as ctx:
        ctx.eval(dw.x, dw.y, dw.z, dw.lam)
        ran.append("eval 1030x3 (row segments)")

    # the fused Nelder-Mead kernel, both shapes, and two batches
    c2 = workloads.config2()
    big, _ = c2.seeded_subset(1500, seed_offset=3)
    small, _ = c2.seeded_subset(48, seed_offset=7)
    with dbie.DBIE.from_workload(c2) as ctx:
        db, ds = dbie.to_device(big), dbie.to_device(small)
        s = ctx.solve(db.x, db.y, db.z)
        ran.append(f"NM 1500 points: {int(s['iters'].sum())} iterations, status counts "
                   f"{np.bincount(s['status'].cpu().numpy(), minlength=4).tolist()}")
        ctx.solve(ds.x, ds.y, ds.z)
        ctx.solve(ds.x, ds.y, ds.z, dbie.default_opts(analytic=1))
        ctx.set_batch_limit(1000)
        s2 = ctx.solve(db.x, db.y, db.z)
        assert torch.equal(s2["lam"], s["lam"])
        ctx.set_batch_limit(0)
        ran.append("NM 48 points (warp shape), analytic, two batches")
        g = ctx.solve(ds.x, ds.y, ds.z, dbie.default_opts(method=1, n_level=3))
        ctx.solve(ds.x, ds.y, ds.z, dbie.default_opts(method=1, n_level=2, n_trial=4, analytic=1))
        ran.append(f"GRID 48 points: levels {int(g['iters'].max())}")
        # tracing: lambda solved at every stage point (field lines), fixed lambda (current lines)
        seeds = [t(a) for a in (np.array([-0.2, 0.25]), np.array([0.1, -0.15]), np.array([0.12, 0.2]))]
        tr = ctx.trace(*seeds, dbie.default_trace_opts(max_steps=3, ds=0.5))
        ctx.trace(*seeds, dbie.default_trace_opts(max_steps=3, current=1, lam=(0.5, 0.5, 0.5)))
        ran.append(f"trace 2 seeds: npts {tr['npts'].cpu().numpy().tolist()}")
    torch.cuda.synchronize()
    print("sanitizer_target ok: " + "; ".join(ran))


if __name__ == "__main__":
    main()
