"""Multi-GPU host logic on CPU: world_size-2 gloo processes shard the points, each
rank computes its shard (the CPU oracle stands in for the per-rank dbie_eval, which needs a GPU),
the shards are gathered back and compared with the unsharded result; timing/work reduction is the
bench contract's max / sum.  No data-path collective exists inside eval/solve."""
import os
import socket

import numpy as np
import pytest

from paper_1306_1122_b200 import sharding


def test_shards_partition_the_points():
    for M in (0, 1, 2, 7, 64, 1000003):
        for world in (1, 2, 3, 8):
            for mode in sharding.MODES:
                if M > 10000 and world > 3:
                    continue
                parts = [sharding.shard_indices(M, r, world, mode) for r in range(world)]
                allidx = np.concatenate(parts)
                assert allidx.size == M and np.array_equal(np.sort(allidx), np.arange(M))
                sizes = [p.size for p in parts]
                assert max(sizes) - min(sizes) <= 1
                assert sizes == sharding.shard_sizes(M, world, mode)
    with pytest.raises(ValueError):
        sharding.shard_indices(10, 2, 2)
    with pytest.raises(ValueError):
        sharding.shard_indices(10, 0, 2, mode="random")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, mode, q):
    import torch
    import torch.distributed as dist
    import oracle
    import workloads
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = workloads.random_boundary(24, 17, seed=5, npts=41, h=0.5)
        # the boundary lives on rank 0 and is replicated by one broadcast
        bx, by, bz = [torch.from_numpy(a.copy()) if rank == 0 else torch.zeros(a.shape, dtype=torch.float64)
                      for a in (w.bx, w.by, w.bz)]
        sharding.broadcast_boundary(dist, bx, by, bz)
        assert np.array_equal(bx.numpy(), w.bx) and np.array_equal(bz.numpy(), w.bz)
        idx = sharding.shard_indices(w.M, rank, world, mode)
        sub = w.subset(idx)
        local = torch.from_numpy(oracle.eval(sub, nthreads=1))               # [3, m_rank]
        full = sharding.gather_points(dist, local, w.M, mode)
        ids = sharding.gather_points(dist, torch.from_numpy(idx.copy()), w.M, mode)
        ms, work = sharding.reduce_over_ranks(dist, "cpu", 10.0 + rank, float(idx.size))
        q.put((rank, full.numpy(), ids.numpy(), ms, work))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("mode", sharding.MODES)
def test_world2_gloo_shard_gather_reduce(mode):
    import torch.multiprocessing as mp
    import oracle
    import workloads
    oracle.build()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, mode, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = [q.get(timeout=240) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = workloads.random_boundary(24, 17, seed=5, npts=41, h=0.5)
    ref = oracle.eval(w, nthreads=1)
    for rank, full, ids, ms, work in got:
        assert np.array_equal(ids, np.arange(w.M))
        assert np.array_equal(full, ref)          # same code per point: bit-identical after the gather
        assert ms == 11.0 and work == float(w.M)  # max over ranks, sum over ranks
