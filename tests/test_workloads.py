"""Seeded input generators (paper_1803_08320_b200/workloads.py): determinism, shapes and
that the closed forms used to SHAPE inputs agree with the paper's printed values (CPU only)."""
import math
import os

import numpy as np

from paper_1803_08320_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def test_splitmix_is_counter_based_and_uniform():
    a = W.splitmix_uniform(42, np.arange(100000))
    b = W.splitmix_uniform(42, np.arange(50000, 100000))
    assert np.array_equal(a[50000:], b)
    assert 0.0 <= a.min() and a.max() < 1.0
    assert abs(a.mean() - 0.5) < 5e-3 and abs(a.var() - 1 / 12) < 2e-3
    assert not np.array_equal(a[:100], W.splitmix_uniform(43, np.arange(100)))


def test_bpt_isco_matches_tables_1_and_2():
    """Tables 1-2; the a=0.9 co-rotating row is last-digit noise in the paper."""
    with open(os.path.join(GOLDEN, "isco_tables.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            sense, a, r, _, _ = [float(x) for x in line.split()]
            tol = 5e-11 if not (a == 0.9 and sense > 0) else 5e-11
            assert abs(W.bpt_isco(1.0, a, sense > 0) - r) < tol, (sense, a)
    assert abs(W.bpt_isco(1.0, 0.0) - 6.0) < 1e-14          # eq.(37)
    assert W.horizon_radius(1.0, 0.0) == 2.0


def test_circular_schwarzschild_config1():
    st = W.circular_schwarzschild(256)
    assert st.shape == (6, 256) and st.flags.c_contiguous
    assert st[0].min() >= 6.5 and st[0].max() <= 20.0
    assert np.allclose(st[5] ** 2, st[0] ** 2 / (st[0] - 3.0))     # eq.(35)
    assert np.array_equal(st, W.circular_schwarzschild(256))


def test_kerr_bound_chunk_independent_and_valid():
    a = 0.9
    s1, c1 = W.kerr_bound(500, a, W.SEED_BASE + 2, chunk=1 << 12, return_constants=True)
    s2 = W.kerr_bound(300, a, W.SEED_BASE + 2, chunk=1 << 15)
    assert np.array_equal(s1[:, :300], s2)
    E, Lz, Q = c1
    assert np.all((E >= 0.9) & (E <= 0.98)) and np.all(np.abs(Lz) <= 4) and np.all((Q >= 0) & (Q <= 12))
    r, th = s1[0], s1[1]
    assert np.all(r >= 1.2 * W.bpt_isco(1.0, a)) and np.all(r <= 30.0)
    assert np.all((th >= math.pi / 6) & (th <= 5 * math.pi / 6))
    # Theta(theta0) = u_theta^2 >= 0 and the drawn Q is recovered from (theta, u_theta)
    Qback = s1[4] ** 2 + np.cos(th) ** 2 * (a * a * (1 - E * E) + Lz ** 2 / np.sin(th) ** 2)
    assert np.allclose(Qback, Q, rtol=1e-10, atol=1e-10)


def test_camera_rays_layout():
    st, (al, be, Lz, Q) = W.camera_rays(8, 0.998, 60.0, return_constants=True)
    assert st.shape == (6, 64)
    assert np.all(st[0] == 1000.0) and np.allclose(st[1], math.radians(60.0))
    assert al[0] == -8.75 and al[7] == 8.75 and be[0] == -8.75 and be[63] == 8.75
    assert np.all(st[3] < 0)                                   # incoming
    tile = W.camera_rays(8, 0.998, 60.0, row0=2, rows=3)
    assert np.array_equal(tile, st[:, 16:40])


def test_shard_range_partitions():
    for n, w in ((10, 3), (4194304, 8), (5, 8), (0, 2)):
        spans = [W.shard_range(n, r, w) for r in range(w)]
        assert spans[0][0] == 0 and spans[-1][1] == n
        assert all(spans[i][1] == spans[i + 1][0] for i in range(w - 1))
        sizes = [hi - lo for lo, hi in spans]
        assert max(sizes) - min(sizes) <= 1
