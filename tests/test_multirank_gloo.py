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


def _bench_worker(rank, world, port, tmpdir):
    """The N > 1 legs of bench.py itself -- dist_init, the MAX/SUM reductions, the strong-scaling shard, the rank-0 JSON
    line, dist_finish -- with the environment torchrun would set, on gloo with CPU tensors standing in for the device."""
    sys.path.insert(0, ROOT)
    import argparse
    import json
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    import torch
    import bench
    from paper_1803_08320_b200 import workloads as W
    dist = bench.dist_init(world, "gloo")
    assert dist is not None and dist.get_world_size() == world
    bench.dist_barrier(dist)
    # weak scaling: every rank reports its own batch; strong: one 64 x 64 image in interleaved row tiles
    img = {"st": W.camera_rays(64, 0.998, 60.0), "name": "test image"}
    mine = bench.shard_for_rank(img, rank, world, "strong")
    rows = 64 // 16
    tiles = W.interleaved_tiles(16, rank, world)
    assert mine["st"].shape[1] == len(tiles) * rows * 64
    assert np.array_equal(mine["st"][:, : rows * 64], img["st"][:, tiles[0] * rows * 64:(tiles[0] + 1) * rows * 64])
    assert bench.shard_for_rank(img, rank, world, "weak") is img
    units = float(mine["st"].shape[1]) * 10.0                       # stand-in: 10 steps per ray
    tmax, tot = bench.reduce_time_and_units(dist, torch.device("cpu"), 100.0 + 50.0 * rank, units)
    assert tmax == 100.0 + 50.0 * (world - 1) and tot == 64 * 64 * 10.0
    if rank == 0:
        args = argparse.Namespace(steps=1, warmup=0)
        line = bench.make_line(args, world, tot / (tmax * 1e-3), tmax, "strong", {"workload": mine["name"]}, {"sm_mhz": None},
                               None, 1, {"bound": "alu"}, None)
        txt = json.dumps(line)
        back = json.loads(txt)
        assert back["n_gpus"] == world and back["scaling"] == "strong" and back["value"] == 64 * 64 * 10.0 / 0.15
        for key in ("metric", "unit", "ms_per_step", "higher_is_better", "vs_baseline", "dtype", "data", "config", "clocks",
                    "e2e", "gpu_launches", "roofline", "cpu_baseline"):
            assert key in back, key
    bench.dist_finish(dist)
    assert not torch.distributed.is_initialized()
    open(os.path.join(tmpdir, f"bench_ok{rank}"), "w").write("ok")


def test_bench_py_multi_rank_legs_on_gloo(tmp_path):
    import socket
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mp.spawn(_bench_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    assert (tmp_path / "bench_ok0").exists() and (tmp_path / "bench_ok1").exists()


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
