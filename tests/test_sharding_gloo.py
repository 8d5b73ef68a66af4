"""world_size-2 `gloo` tests (CPU) of the multi-GPU plumbing: view sharding, unit / timing reductions, the
volume all-reduce of a view-sharded back-projection and the per-view gather.  The data path itself has no
collective; the arithmetic that stands in for the kernels here is the fp64 oracle,
which is linear in exactly the way the sharding relies on (Eq.21 is a sum over views)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2508_13304_b200.sharding import (allreduce_volume, gather_view_results, job_throughput, max_over_ranks,
                                            shard_range, sum_over_ranks)


def test_shard_range_tiles_and_balances():
    for n in (0, 1, 5, 64, 360, 721):
        for world in (1, 2, 3, 8):
            parts = [shard_range(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    import sys
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    import oracle
    from helpers import small_geom
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # reductions
        t = max_over_ranks(torch.tensor([1.0 + rank, 5.0 - rank], dtype=torch.float64))
        assert t.tolist() == [float(world), 5.0]
        u = sum_over_ranks(torch.tensor([10.0 * (rank + 1)], dtype=torch.float64))
        assert u.item() == 10.0 * world * (world + 1) / 2
        rate, units, secs = job_throughput(100.0 * (rank + 1), 2.0 + rank)
        assert units == 100.0 * world * (world + 1) / 2 and secs == 1.0 + world and rate == units / secs
        # view-sharded back-projection == full back-projection after the volume all-reduce
        g = small_geom(n=10, nu=12, nv=9)
        V = 5
        rng = np.random.default_rng(7)
        angles = rng.uniform(0, 6.28, V)
        poses = rng.uniform(-0.1, 0.1, (V, 6))
        proj = rng.standard_normal((V,) + g.det_shape).astype(np.float32)
        lo, hi = shard_range(V, rank, world)
        part = torch.from_numpy(oracle.backproject(g, angles[lo:hi], poses[lo:hi], proj[lo:hi]))
        full = allreduce_volume(part)
        ref = oracle.backproject(g, angles, poses, proj)
        assert np.allclose(full.numpy(), ref, rtol=1e-12, atol=1e-14)
        # per-view results gathered in view order (uneven shards: 3 + 2)
        vol = rng.standard_normal(g.vol_shape).astype(np.float32)
        up = rng.standard_normal((V,) + g.det_shape).astype(np.float32)
        local = torch.from_numpy(oracle.forward_pose_grad(g, angles[lo:hi], poses[lo:hi], vol, up[lo:hi]))
        allg = gather_view_results(local, V)
        refg = oracle.forward_pose_grad(g, angles, poses, vol, up)
        assert allg.shape == (V, 6) and np.array_equal(allg.numpy(), refg)
        open(os.path.join(out_dir, f"ok{rank}"), "w").write("ok")
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert all((tmp_path / f"ok{r}").exists() for r in range(world))
