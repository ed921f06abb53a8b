"""Helpers of the GPU tests: run the CUDA path through the binding, compare snapshot buffers."""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import parity  # noqa: E402


def run_gpu(G, metric, a, st, h, nsteps, flags=0, snapshot_every=0, snap_mask=0xFF, snap_capacity=None,
            host=False, M=1.0, **stop):
    import torch
    ctx = G.geo_create(metric, M, a)
    try:
        n = st.shape[1]
        if host:
            out = G.alloc_outputs_host(n, nsteps, snapshot_every, snap_capacity, snap_mask)
            G.geo_integrate_host(ctx, np.ascontiguousarray(st), h, nsteps, out, flags=flags,
                                 snapshot_every=snapshot_every, **stop)
            return G.to_numpy(out)
        dev = torch.device("cuda:0")
        d_in = torch.from_numpy(np.ascontiguousarray(st)).to(dev)
        out = G.alloc_outputs(n, dev, nsteps, snapshot_every, snap_capacity, snap_mask)
        G.geo_integrate(ctx, d_in, h, nsteps, out, flags=flags, snapshot_every=snapshot_every, **stop)
        torch.cuda.synchronize()
        return G.to_numpy(out)
    finally:
        G.geo_destroy(ctx)


def assert_snapshots_match(g, o, tol):
    assert np.array_equal(g["snap_count"], o["snap_count"])
    cap = o["snapshots"].shape[1]
    valid = np.arange(cap)[None, :] < np.minimum(o["snap_count"], cap)[:, None]
    e = parity.rel_err(g["snapshots"], o["snapshots"])
    assert e[valid].max() <= tol, e[valid].max()
    # slots >= snap_count are left untouched (NaN-filled by the allocator on both sides)
    assert np.isnan(g["snapshots"][~valid]).all()
