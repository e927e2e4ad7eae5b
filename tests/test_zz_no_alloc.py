"""dbie_eval_noalloc: the eval entry point for callers that cannot allocate device memory.

Some programs that would embed this library cannot let it call cudaMalloc: a framework that gives all of
HBM to its own memory pool when it starts (a later cudaMalloc then simply fails), or a time-stepping loop
in which the device-wide synchronisation of cudaMalloc / cudaFree is not acceptable.  dbie_eval obtains its
partial-sum buffer with cudaMalloc on first use; dbie_eval_noalloc keeps those sums in a fixed 6 MiB array
inside the library instead and therefore takes at most 16,384 points per call (include/dbie.h).

The test compares it with the existing path (DBIE.eval -> dbie_eval) on the same inputs, on two calls in a
row that share the array (the second smaller, with other lambda and another boundary, so that stale partial
sums of the first would show), at the parity tolerance of the other GPU tests (1e-9 relative) and, since both
run the same kernels in the same summation order, bit for bit.

The file name sorts after every other test file on purpose: `pytest -x` stops at the first failure, and a
failure here must not hide the parity tests.  Nothing here depends on what ran before it.
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

TOL_B = 1e-9   # tests/test_gpu_parity.py's bound on max_i ||dB_i|| / ||B_i||


@pytest.fixture(scope="module")
def dbie():
    import torch
    assert torch.cuda.is_available()
    import paper_1306_1122_b200 as d
    d.load()     # raises if the CUDA library is missing: no fallback
    return d


def _relerr(B, R):
    n = np.linalg.norm(R, axis=0)
    keep = n >= 1e-6 * n.max()
    return float((np.linalg.norm(B - R, axis=0)[keep] / n[keep]).max())


def test_two_calls_in_a_row_match_dbie_eval(dbie):
    import torch
    limit = dbie.noalloc_max_points()
    assert limit == 16384
    # call 1: a 96 x 80 boundary (16 chunks of 5 rows), 5,001 points (19 full blocks of 256 and a tail of 137)
    w1 = workloads.random_boundary(96, 80, seed=101, npts=5001, h=0.7, x0=-3.0, y0=1.5)
    w1.lam[:, 0] = 0.0
    w1.lam[2, 1] = -w1.lam[2, 1]
    # call 2: another boundary with fewer chunks (7 rows -> 7 chunks) and fewer points, other lambda
    w2 = workloads.random_boundary(600, 7, seed=202, npts=777, h=0.5, x0=0.0, y0=-2.0)
    with dbie.DBIE.from_workload(w1) as c1, dbie.DBIE.from_workload(w2) as c2:
        d1, d2 = dbie.to_device(w1), dbie.to_device(w2)
        out1 = torch.full((3, w1.M), float("nan"), dtype=torch.float64, device="cuda")
        out2 = torch.full((3, w2.M), float("nan"), dtype=torch.float64, device="cuda")
        # the two calls in a row on the shared array, same stream, nothing in between
        c1.eval_noalloc(d1.x, d1.y, d1.z, d1.lam, out1)
        c2.eval_noalloc(d2.x, d2.y, d2.z, d2.lam, out2)
        ref1 = c1.eval(d1.x, d1.y, d1.z, d1.lam)          # the existing path
        ref2 = c2.eval(d2.x, d2.y, d2.z, d2.lam)
        torch.cuda.synchronize()
        for out, ref in ((out1, ref1), (out2, ref2)):
            assert bool(torch.isfinite(out).all())
            assert _relerr(out.cpu().numpy(), ref.cpu().numpy()) <= TOL_B
            assert torch.equal(out, ref)                  # same kernels, same chunk order: bit-identical
        # a third call re-using context 1 after context 2 wrote the array: still the same bits
        out1.fill_(float("nan"))
        c1.eval_noalloc(d1.x, d1.y, d1.z, d1.lam, out1)
        assert torch.equal(out1, ref1)
        assert c1.counters()["interactions"] == float(w1.M) * w1.N


def test_exactly_the_limit_and_one_more(dbie):
    import torch
    limit = dbie.noalloc_max_points()
    w = workloads.random_boundary(33, 17, seed=303, npts=limit + 1, h=1.0, x0=0.0, y0=0.0)
    with dbie.DBIE.from_workload(w) as ctx:
        d = dbie.to_device(w)
        out = torch.empty((3, w.M), dtype=torch.float64, device="cuda")
        with pytest.raises(dbie.DBIEError) as ei:         # one point too many: refused before any launch
            ctx.eval_noalloc(d.x, d.y, d.z, d.lam, out)
        assert ei.value.status == dbie.DBIE_EINVAL
        assert "DBIE_NOALLOC_MAX_POINTS" in str(ei.value) and str(limit) in str(ei.value)
        # exactly the limit fills the whole array and is accepted
        sub = w.subset(np.arange(limit))
        ds = dbie.to_device(sub)
        out = torch.empty((3, limit), dtype=torch.float64, device="cuda")
        ctx.eval_noalloc(ds.x, ds.y, ds.z, ds.lam, out)
        assert torch.equal(out, ctx.eval(ds.x, ds.y, ds.z, ds.lam))
        # M = 0 is a no-op
        e = torch.empty((0,), dtype=torch.float64, device="cuda")
        ctx.eval_noalloc(e, e, e, torch.empty((3, 0), dtype=torch.float64, device="cuda"),
                         torch.empty((3, 0), dtype=torch.float64, device="cuda"))
