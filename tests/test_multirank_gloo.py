"""N > 1 host-side logic on CPU: world_size-2 `gloo` run of the sharding bench.py uses under torchrun.

The path shards with no exchange step (geodesics are independent):
each rank integrates its own contiguous index range (or its interleaved image tiles) and the only
collectives are the bench's reductions (SUM of steps, MAX of time).  Here each rank's "device" is the
CPU oracle (test infrastructure), so the test checks the partition + reductions, not a kernel.
"""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, tmpdir):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import torch
    import torch.distributed as dist
    import geo_oracle
    from paper_1803_08320_b200 import workloads as W

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # (1) contiguous shards of a timelike batch
        n, a = 301, 0.9
        full = W.kerr_bound(n, a, W.SEED_BASE + 2)
        lo, hi = W.shard_range(n, rank, world)
        mine = np.ascontiguousarray(full[:, lo:hi])
        o = geo_oracle.integrate(geo_oracle.KERR, 1.0, a, mine, 0.01, 200)
        steps = torch.tensor([float(o["steps_done"].sum())], dtype=torch.float64)
        tmax = torch.tensor([1.0 + rank], dtype=torch.float64)        # stand-in for the per-rank event time
        dist.all_reduce(steps, op=dist.ReduceOp.SUM)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        assert steps.item() == 200.0 * n and tmax.item() == float(world)
        # gather the final states on rank 0 (the optional "results on one device" step of SURVEY 8(e))
        sizes = [W.shard_range(n, r, world) for r in range(world)]
        pad = max(h - l for l, h in sizes)
        buf = torch.zeros((8, pad), dtype=torch.float64)
        buf[:, : hi - lo] = torch.from_numpy(o["final_state"])
        got = [torch.zeros_like(buf) for _ in range(world)]
        dist.all_gather(got, buf)
        if rank == 0:
            whole = geo_oracle.integrate(geo_oracle.KERR, 1.0, a, full, 0.01, 200)["final_state"]
            cat = np.concatenate([g.numpy()[:, : h - l] for g, (l, h) in zip(got, sizes)], axis=1)
            assert np.array_equal(cat, whole)          # sharding does not change a single bit
        # (2) interleaved row tiles of a camera image
        N, rows = 16, 4
        tiles = W.interleaved_tiles(N // rows, rank, world)
        cnt = torch.tensor([float(len(tiles))])
        dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
        assert cnt.item() == N // rows
        img = W.camera_rays(N, 0.998, 60.0)
        for t in tiles:
            assert np.array_equal(W.camera_rays(N, 0.998, 60.0, row0=t * rows, rows=rows), img[:, t * rows * N:(t + 1) * rows * N])
        open(os.path.join(tmpdir, f"ok{rank}"), "w").write("ok")
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_sharding(tmp_path):
    import socket
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    assert (tmp_path / "ok0").exists() and (tmp_path / "ok1").exists()


def test_interleaved_tiles_cover_once():
    from paper_1803_08320_b200 import workloads as W
    for nt, w in ((16, 8), (16, 3), (1, 2)):
        allt = sorted(t for r in range(w) for t in W.interleaved_tiles(nt, r, w))
        assert allt == list(range(nt))
