"""GPU edge cases and invariants of the C-ABI path: empty / single / ragged batches, degenerate stop
cases (B1), capacity overflow (S3), backwards integration, host-buffer entry point, queue vs static
mapping, argument errors.  Each compares with the oracle or with a property that holds at any size."""
import math
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import parity  # noqa: E402
from gpu_helpers import run_gpu, assert_snapshots_match  # noqa: E402

from paper_1803_08320_b200 import workloads as W  # noqa: E402

pytestmark = pytest.mark.gpu


def test_empty_batch_is_ok_and_launches_nothing(G):
    import torch
    ctx = G.geo_create(G.KERR, 1.0, 0.5)
    d_in = torch.empty((6, 0), dtype=torch.float64, device="cuda:0")
    out = G.alloc_outputs(0, d_in.device)
    G.geo_integrate(ctx, d_in, 0.01, 10, out)
    torch.cuda.synchronize()
    G.geo_destroy(ctx)


@pytest.mark.parametrize("n", [1, 31, 33, 129])
def test_tiny_and_ragged_batches(G, oracle, n):
    st = W.kerr_bound(n, 0.9, W.SEED_BASE + 2)
    o = oracle.integrate(oracle.KERR, 1.0, 0.9, st, 0.01, 500)
    for flags in (0, G.FLAG_STATIC_MAP):
        g = run_gpu(G, G.KERR, 0.9, st, 0.01, 500, flags=flags)
        c = parity.compare(g, o)
        assert c["same_class"].all() and c["err"].max() <= 1e-9


def test_degenerate_stop_cases_B1(G, oracle):
    """y0 already inside r_capture -> CAPTURED, 0 steps, no slot 0; y0 beyond r_escape -> ESCAPED with
    slot 0; nsteps = 0 -> MAXSTEPS; NaN input -> NUMERIC."""
    st = W.kerr_bound(8, 0.5, W.SEED_BASE + 4)
    st[0, 0] = 1.5      # < r_capture
    st[0, 1] = 500.0    # > r_escape
    st[3, 2] = np.nan   # non-finite momentum
    kw = dict(r_capture=2.0, r_escape=100.0, snapshot_every=5)
    o = oracle.integrate(oracle.KERR, 1.0, 0.5, st, 0.01, 20, **kw)
    g = run_gpu(G, G.KERR, 0.5, st, 0.01, 20, **kw)
    assert np.array_equal(g["status"], o["status"]) and np.array_equal(g["steps_done"], o["steps_done"])
    assert g["status"][0] == G.ST_CAPTURED and g["status"][1] == G.ST_ESCAPED and g["status"][2] == G.ST_NUMERIC
    assert np.array_equal(g["snap_count"], o["snap_count"])
    assert g["snap_count"][0] == 0 and g["snap_count"][1] == 1
    ok = np.ones(8, bool)
    ok[2] = False
    assert parity.rel_err(g["final_state"], o["final_state"])[:, ok].max() <= 1e-12
    o0 = oracle.integrate(oracle.KERR, 1.0, 0.5, st[:, 3:], 0.01, 0)
    g0 = run_gpu(G, G.KERR, 0.5, st[:, 3:], 0.01, 0)
    assert (g0["status"] == G.ST_MAXSTEPS).all() and (g0["steps_done"] == 0).all()
    assert parity.rel_err(g0["final_state"], o0["final_state"]).max() <= 1e-15


def test_capture_keeps_last_accepted_state(G, oracle):
    """B2: plunging timelike particles (r < r_isco, E and L of a slightly sub-circular orbit) are
    CAPTURED at the guard; final state has r >= r_capture and is finite; class equals the oracle's."""
    n = 64
    st = np.zeros((6, n))
    st[0] = np.linspace(3.2, 5.5, n)
    st[1] = math.pi / 2
    st[3] = -0.05
    st[5] = 0.9 * st[0] * np.sqrt(1.0 / (st[0] - 3.0))
    kw = dict(r_capture=2.0 + 1e-3, r_escape=50.0)
    o = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, st, 0.01, 20000, **kw)
    g = run_gpu(G, G.SCHWARZSCHILD, 0.0, st, 0.01, 20000, **kw)
    c = parity.compare(g, o)
    assert (o["status"] == oracle.ST_CAPTURED).all()
    assert c["same_class"].all() and c["err"].max() <= 1e-9
    assert (g["final_state"][1] >= 2.0 + 1e-3).all() and np.isfinite(g["final_state"]).all()


def test_snapshot_capacity_overflow_drops_but_counts_S3(G, oracle):
    st = W.circular_schwarzschild(40)
    for mask, flags in ((0xFF, 0), (0x0E, 0), (0x07, 0), (0xFF, G.FLAG_STAGED_SNAP), (0x07, G.FLAG_STAGED_SNAP), (0x0F, G.FLAG_STAGED_SNAP)):   # 0x07: odd ncomp
        o = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, st, 0.01, 100, snapshot_every=7, snap_capacity=6, snap_mask=mask)
        g = run_gpu(G, G.SCHWARZSCHILD, 0.0, st, 0.01, 100, snapshot_every=7, snap_capacity=6, snap_mask=mask, flags=flags)
        assert (g["snap_count"] == 1 + 100 // 7).all()
        assert_snapshots_match(g, o, 1e-9)


def test_snapshot_slot_equals_shorter_run_bitwise(G):
    """SURVEY 8(c) pin 'Snapshots': slot j equals the final state of a run with nsteps = j*snapshot_every."""
    st = W.kerr_bound(200, 0.9, W.SEED_BASE + 2)
    g = run_gpu(G, G.KERR, 0.9, st, 0.01, 300, snapshot_every=100)
    for j in (1, 2, 3):
        gj = run_gpu(G, G.KERR, 0.9, st, 0.01, 100 * j)
        assert np.array_equal(g["snapshots"][:, j, :], gj["final_state"].T)


def test_backwards_integration_returns_to_start(G, oracle):
    """h < 0 is legal; forward then backward with RK4 returns to y0 up to O(h^4) truncation."""
    st = W.kerr_bound(64, 0.5, W.SEED_BASE + 4)
    o = oracle.integrate(oracle.KERR, 1.0, 0.5, st, -0.01, 1000)
    g = run_gpu(G, G.KERR, 0.5, st, -0.01, 1000)
    c = parity.compare(g, o)
    assert c["same_class"].all() and c["err"].max() <= 1e-9
    back_in = np.ascontiguousarray(g["final_state"][[1, 2, 3, 5, 6, 7]])
    b = run_gpu(G, G.KERR, 0.5, back_in, 0.01, 1000)
    assert np.abs(b["final_state"][[1, 2, 5, 6]] - st[[0, 1, 3, 4]]).max() < 1e-8


def test_host_entry_point_is_bitwise_equal_to_device_entry_point(G):
    st = W.kerr_bound(777, 0.9, W.SEED_BASE + 2)
    kw = dict(snapshot_every=50, snap_mask=0x3F)
    a = run_gpu(G, G.KERR, 0.9, st, 0.01, 400, **kw)
    b = run_gpu(G, G.KERR, 0.9, st, 0.01, 400, host=True, **kw)
    for k in ("final_state", "status", "steps_done", "eq_cross_r", "health", "snapshots", "snap_count"):
        assert np.array_equal(a[k], b[k], equal_nan=True), k


def test_host_entry_point_chunked_pipeline_is_bitwise_equal(G):
    """A job above the host path's chunk threshold (1.05 GB of snapshots, 400 003 particles -> two
    double-buffered chunks, ragged last chunk) returns what the one-launch device path returns."""
    st = W.circular_schwarzschild(400003, W.SEED_BASE + 7)
    kw = dict(snapshot_every=1, snap_mask=0xFF)
    a = run_gpu(G, G.SCHWARZSCHILD, 0.0, st, 0.01, 40, **kw)
    b = run_gpu(G, G.SCHWARZSCHILD, 0.0, st, 0.01, 40, host=True, **kw)
    for k in ("final_state", "status", "steps_done", "eq_cross_r", "health", "snapshots", "snap_count"):
        assert np.array_equal(a[k], b[k], equal_nan=True), k
    assert (b["snap_count"] == 41).all() and not np.isnan(b["snapshots"]).any()


def test_queue_and_static_mapping_and_reruns_are_bitwise_identical(G):
    """No arithmetic crosses lanes: results do not depend on which lane integrated a particle."""
    a = 0.998
    st, _ = W.camera_rays(64, a, 60.0, return_constants=True)
    st = np.ascontiguousarray(st[:, ::3])
    kw = dict(r_capture=W.horizon_radius(1.0, a) + 0.01, r_escape=1100.0, kind=G.NULL)
    ref = run_gpu(G, G.KERR, a, st, 0.02, 200000, **kw)
    for flags in (0, G.FLAG_STATIC_MAP):
        g = run_gpu(G, G.KERR, a, st, 0.02, 200000, flags=flags, **kw)
        for k in ("final_state", "status", "steps_done", "eq_cross_r"):
            assert np.array_equal(ref[k], g[k], equal_nan=True), (flags, k)


def test_plain_update_flag_matches_oracle_plain(G, oracle):
    st = W.kerr_bound(128, 0.9, W.SEED_BASE + 2)
    o = oracle.integrate(oracle.KERR, 1.0, 0.9, st, 0.01, 2000, flags=oracle.FLAG_PLAIN_UPDATE)
    g = run_gpu(G, G.KERR, 0.9, st, 0.01, 2000, flags=G.FLAG_PLAIN_UPDATE)
    c = parity.compare(g, o)
    assert c["same_class"].all() and c["err"].max() <= 1e-9


def test_argument_errors_return_einval_without_launch(G):
    import torch
    ctx = G.geo_create(G.KERR, 1.0, 0.5)
    d_in = torch.zeros((6, 4), dtype=torch.float64, device="cuda:0")
    out = G.alloc_outputs(4, d_in.device)
    for kw in (dict(h=0.0), dict(h=float("nan")), dict(nsteps=-1), dict(kind=7), dict(flags=64),
               dict(snapshot_every=5)):                        # snapshots NULL
        args = dict(h=0.01, nsteps=10)
        args.update(kw)
        with pytest.raises(G.GeoError) as ei:
            G.geo_integrate(ctx, d_in, args.pop("h"), args.pop("nsteps"), out, **args)
        assert ei.value.code == G.EINVAL and G.geo_last_error(ctx)
    mis = torch.zeros(6 * 4 + 1, dtype=torch.float64, device="cuda:0")[1:].view(6, 4)   # 8-byte aligned only
    with pytest.raises(G.GeoError):
        G.geo_integrate(ctx, mis, 0.01, 10, out)
    G.geo_destroy(ctx)
    for bad in ((G.KERR, 1.0, 1.5), (G.SCHWARZSCHILD, 1.0, 0.1), (5, 1.0, 0.0), (G.KERR, -1.0, 0.0)):
        with pytest.raises(G.GeoError):
            G.geo_create(*bad)
    ctx = G.geo_create(G.KERR, 1.0, 0.6)
    assert G.geo_horizon_radius(ctx) == 1.0 + math.sqrt(1.0 - 0.36)
    G.geo_destroy(ctx)


def test_mass_and_negative_spin(G, oracle):
    """M != 1 and a < 0 through the CUDA path: parity with the oracle and the exact M-scaling symmetry of the
    metric (lengths, t, L, p_theta scale with M) against the M = 1 CUDA result."""
    a, M = 0.7, 2.5
    st = W.kerr_bound(500, a, W.SEED_BASE + 2)
    sM = st.copy()
    sM[0] *= M
    sM[4] *= M
    sM[5] *= M
    g1 = run_gpu(G, G.KERR, a, st, 0.01, 3000, r_capture=2.0, r_escape=100.0)
    gM = run_gpu(G, G.KERR, a * M, sM, 0.01 * M, 3000, M=M, r_capture=2.0 * M, r_escape=100.0 * M)
    oM = oracle.integrate(oracle.KERR, M, a * M, sM, 0.01 * M, 3000, r_capture=2.0 * M, r_escape=100.0 * M, nthreads=8)
    c = parity.compare(gM, oM)
    assert c["same_class"].all() and c["err"].max() <= 1e-9
    scale = np.array([M, M, 1, 1, 1, 1, M, M])[:, None]
    assert np.max(np.abs(gM["final_state"] / scale - g1["final_state"]) / np.maximum(np.abs(g1["final_state"]), 1)) < 1e-10
    flip = st.copy()
    flip[5] *= -1.0
    gf = run_gpu(G, G.KERR, -a, flip, 0.01, 3000, r_capture=2.0, r_escape=100.0)
    of = oracle.integrate(oracle.KERR, 1.0, -a, flip, 0.01, 3000, r_capture=2.0, r_escape=100.0, nthreads=8)
    c = parity.compare(gf, of)
    assert c["same_class"].all() and c["err"].max() <= 1e-9
    sign = np.array([1, 1, 1, -1, 1, 1, 1, -1])[:, None]
    assert np.max(np.abs(gf["final_state"] * sign - g1["final_state"])) < 1e-10


def test_small_batch_instantiation_gives_the_bits_of_the_full_machine_one(G):
    """Batches without records that fit on the machine at 2 CTAs per SM (n <= 37 888) run the WIDE instantiation of the
    kernel (more registers, more instructions in flight per warp: such a batch is latency-bound); same source, same
    arithmetic: a particle's result must not depend on which instantiation integrated it."""
    a = 0.998
    big = W.camera_rays(256, a, 60.0)                             # 65 536 rays: the 128-register instantiation
    ii = np.arange(0, 65536, 53)                                  # 1 237 of them alone: the wide one
    kw = dict(r_capture=W.horizon_radius(1.0, a) + 0.01, r_escape=1100.0, kind=G.NULL)
    gb = run_gpu(G, G.KERR, a, big, 0.02, 200000, **kw)
    gs = run_gpu(G, G.KERR, a, np.ascontiguousarray(big[:, ii]), 0.02, 200000, **kw)
    for k in ("final_state", "status", "steps_done", "eq_cross_r", "health"):
        assert np.array_equal(gb[k][..., ii], gs[k], equal_nan=True), k
    st = W.kerr_bound(70000, 0.5, W.SEED_BASE + 4)
    tb = run_gpu(G, G.KERR, 0.5, st, 0.01, 300, flags=G.FLAG_PLAIN_UPDATE)
    ts = run_gpu(G, G.KERR, 0.5, np.ascontiguousarray(st[:, :5000]), 0.01, 300, flags=G.FLAG_PLAIN_UPDATE)
    assert np.array_equal(tb["final_state"][:, :5000], ts["final_state"])


@pytest.mark.parametrize("snapshot_every", [0, 100])
def test_one_wave_batches_on_one_cta_per_sm_give_the_same_bits(G, snapshot_every):
    """A batch that fits in one wave (n <= 512 x SMs) runs ONE CTA of 128 k threads per SM, k = ceil(n / (128 SMs))
    (geo_kernel.cuh: BIG; WIDE takes 256).  Same source, same arithmetic: every particle's result -- trajectory records
    included -- is bitwise what it is in a batch of another size class (k = 1, 2, 3, 4 and multi-wave), with the queue and
    with the static mapping."""
    import torch
    sm = torch.cuda.get_device_properties(0).multi_processor_count
    n = sm * 3 * 128 + 1000                                                  # k = 4
    st = W.kerr_bound(n, 0.9, W.SEED_BASE + 2)
    kw = dict(snapshot_every=snapshot_every, snap_mask=0x6F)
    ctx = G.geo_create(G.KERR, 1.0, 0.9)
    try:
        for m, blk in ((n, 512), (sm * 3 * 128, 384), (sm * 2 * 128 + 1, 384), (sm * 128 + 1, 256), (sm * 128, 128), (sm * 512 + 1, 128)):
            info = G.geo_launch_info(ctx, m, 0, snapshot_every)
            assert info["block"] == blk and (blk == 128 or info["grid"] <= sm), (m, info)
        assert G.geo_launch_info(ctx, n, G.FLAG_STAGED_SNAP, 100)["block"] == 128      # the staged writer keeps its 128-thread stage
    finally:
        G.geo_destroy(ctx)
    big = run_gpu(G, G.KERR, 0.9, st, 0.01, 300, **kw)
    big_static = run_gpu(G, G.KERR, 0.9, st, 0.01, 300, flags=G.FLAG_STATIC_MAP, **kw)
    for lo, hi in ((0, 5000), (1000, 1000 + sm * 128 + 77), (n - 45000, n)):        # k = 1, k = 2, k = 3
        small = run_gpu(G, G.KERR, 0.9, np.ascontiguousarray(st[:, lo:hi]), 0.01, 300, **kw)
        for res in (big, big_static):
            assert np.array_equal(res["final_state"][:, lo:hi].view(np.int64), small["final_state"].view(np.int64))
            assert np.array_equal(res["status"][lo:hi], small["status"]) and np.array_equal(res["steps_done"][lo:hi], small["steps_done"])
            assert np.array_equal(res["eq_cross_r"][lo:hi].view(np.int64), small["eq_cross_r"].view(np.int64))
            if snapshot_every:
                assert np.array_equal(res["snap_count"][lo:hi], small["snap_count"])
                assert np.array_equal(res["snapshots"][lo:hi].view(np.int64), small["snapshots"].view(np.int64))
    # multi-wave (128-thread CTAs, queue refill): the first 3000 particles of a 2-wave batch
    nn = sm * 512 + 3000
    st2 = W.kerr_bound(nn, 0.9, W.SEED_BASE + 2)
    assert np.array_equal(st2[:, :n], st)                                        # (the generator is prefix-stable)
    multi = run_gpu(G, G.KERR, 0.9, st2, 0.01, 300, **kw)
    assert np.array_equal(multi["final_state"][:, :n].view(np.int64), big["final_state"].view(np.int64))
