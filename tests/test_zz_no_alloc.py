"""geo_integrate_host_noalloc (include/geo.h): the allocation-free entry point against the existing host path.

The entry point runs the kernels of geo_integrate_host with all device scratch (work-queue head, staging of inputs and
outputs) in a static __device__ array of the library, at most GEO_NOALLOC_MAX_N = 65536 particles per call.  Same
kernel instantiation, same grid, same per-particle arithmetic as the existing path, so the comparison is BITWISE (tighter
than the 1e-9 the parity tests use against the oracle).  The calls run back to back on the shared scratch, a smaller batch
after a larger one, so stale contents of the previous call would show.

Collected last on purpose (file name): the suite runs with pytest -x.
"""
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

from paper_1803_08320_b200 import workloads as W  # noqa: E402

pytestmark = pytest.mark.gpu

KEYS = ("final_state", "status", "steps_done", "eq_cross_r", "health", "coarse_steps")


def _cases(G):
    """(label, metric, a, state, h, nsteps, stop keywords) -- a batch above the WIDE threshold on the Kerr queue kernel, a
    ragged smaller one on the Schwarzschild kernel with the plain update and both stop radii, the maximum size."""
    a = 0.9
    bound = W.kerr_bound(50000, a, W.SEED_BASE + 41)
    rays = W.camera_rays(64, 0.0, 60.0, r_obs=50.0, width=16.0)[:, :3001]
    full = W.kerr_bound(G.NOALLOC_MAX_N, 0.5, W.SEED_BASE + 42)
    return [
        ("kerr_bound_50000", G.KERR, a, bound, 0.05, 400, dict(kind=G.TIMELIKE)),
        ("schw_rays_3001", G.SCHWARZSCHILD, 0.0, rays, 0.05, 3000,
         dict(kind=G.NULL, r_capture=2.0 * 1.001, r_escape=55.0, flags=G.FLAG_PLAIN_UPDATE)),
        ("kerr_bound_max_n", G.KERR, 0.5, full, 0.1, 60, dict(kind=G.TIMELIKE, flags=G.FLAG_STATIC_MAP)),
    ]


def _existing(G, metric, a, st, h, nsteps, kw):
    ctx = G.geo_create(metric, 1.0, a)
    try:
        out = G.alloc_outputs_host(st.shape[1], want_coarse=True)
        G.geo_integrate_host(ctx, np.ascontiguousarray(st), h, nsteps, out, **kw)
        return G.to_numpy(out)
    finally:
        G.geo_destroy(ctx)


def _noalloc(G, metric, a, st, h, nsteps, kw, stream=None):
    out = G.alloc_outputs_host(st.shape[1], want_coarse=True)
    for k in KEYS:                       # poison: every element must be written by the call
        out[k].view(np.uint8)[...] = 0xA5
    G.geo_integrate_host_noalloc(metric, 1.0, a, np.ascontiguousarray(st), h, nsteps, out, stream=stream, **kw)
    return G.to_numpy(out)


def _assert_same_bits(label, g, ref):
    for k in KEYS:
        x, y = np.ascontiguousarray(g[k]), np.ascontiguousarray(ref[k])
        assert x.shape == y.shape and x.dtype == y.dtype, (label, k)
        same = x.view(np.uint8) == y.view(np.uint8)
        assert same.all(), (label, k, int((~same).sum()))


def test_noalloc_matches_existing_path_on_calls_in_a_row(G):
    import torch
    cases = _cases(G)
    ref = [_existing(G, m, a, st, h, ns, kw) for (_, m, a, st, h, ns, kw) in cases]
    # the cases do something: every termination class the stop rules give occurs, and the Kerr batch is above the WIDE threshold
    assert set(np.unique(ref[1]["status"])) >= {G.ST_CAPTURED, G.ST_ESCAPED}
    assert cases[0][3].shape[1] > 148 * 2 * 128
    side = torch.cuda.Stream()
    free = []
    for rnd in range(2):                 # second round: the scratch holds the first round's contents, no memory moved
        torch.cuda.synchronize()
        free.append(torch.cuda.mem_get_info()[0])
        for i, (label, m, a, st, h, ns, kw) in enumerate(cases):
            g = _noalloc(G, m, a, st, h, ns, kw, stream=side if (i + rnd) % 2 else None)
            _assert_same_bits(f"{label} round {rnd}", g, ref[i])
    torch.cuda.synchronize()
    free.append(torch.cuda.mem_get_info()[0])
    # kernels are loaded and the scratch address resolved in round 0; round 1 leaves the device's free memory untouched
    assert free[2] == free[1], free


def test_noalloc_rejects_oversize_and_bad_arguments(G):
    n = G.NOALLOC_MAX_N + 1
    st = np.zeros((6, n))
    st[0] = 10.0
    st[1] = 1.0
    out = G.alloc_outputs_host(n)
    out["status"].fill(-7)
    with pytest.raises(G.GeoError) as ei:
        G.geo_integrate_host_noalloc(G.KERR, 1.0, 0.9, st, 0.1, 10, out)
    assert ei.value.code == G.EINVAL
    assert "GEO_NOALLOC_MAX_N" in str(ei.value) and str(n) in str(ei.value)
    assert (out["status"] == -7).all()                     # nothing was enqueued
    small, o2 = st[:, :8].copy(), G.alloc_outputs_host(8)
    for bad in (dict(metric=G.TABULATED), dict(a=1.5), dict(flags=G.FLAG_STAGED_SNAP), dict(h=0.0)):
        kw = dict(metric=G.KERR, a=0.9, h=0.1, flags=0)
        kw.update(bad)
        with pytest.raises(G.GeoError) as ei:
            G.geo_integrate_host_noalloc(kw["metric"], 1.0, kw["a"], small, kw["h"], 10, o2, flags=kw["flags"])
        assert ei.value.code == G.EINVAL and len(str(ei.value)) > 20, bad
    # and the path still works after the rejected calls
    G.geo_integrate_host_noalloc(G.KERR, 1.0, 0.9, small, 0.1, 10, o2)
    assert (o2["steps_done"] == 10).all() and (o2["status"] == G.ST_MAXSTEPS).all()
