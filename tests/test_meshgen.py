"""The seeded input generator: canonical form, clustering structure, determinism."""
import numpy as np
import pytest

import meshgen


def _check_canonical(m):
    T = m.simplices
    assert T.dtype == np.int32 and T.shape[1] == m.dim + 1
    assert np.all(np.diff(T, axis=1) > 0)                                    # C1
    if len(T) > 1:
        d = np.diff(T.astype(np.int64), axis=0)
        first = np.argmax(d != 0, axis=1)
        assert np.all(d[np.arange(len(d)), first] > 0)                       # C2 strictly ascending rows
    assert T.min() >= 0 and T.max() < m.num_vertices                         # C3
    o = m.cluster_offsets
    assert o[0] == 0 and o[-1] == m.num_vertices and np.all(np.diff(o) >= 0)


def test_config1_exact():
    m = meshgen.make_config(1)
    _check_canonical(m)
    assert (m.num_vertices, m.num_simplices, m.num_clusters) == (4096, 20250, 8)
    assert np.all(np.diff(m.cluster_offsets) == 512)
    # internal simplices per cluster: 2,058 - 3,072
    first = np.searchsorted(m.simplices[:, 0], m.cluster_offsets)
    per = np.diff(first)
    assert per.min() == 2058 and per.max() == 3072


@pytest.mark.parametrize("cfg,n,nC,size", [(2, 256, 16, 4096), (3, 32, 8, 4096), (5, 32, 8, 4096)])
def test_small_configs_structure(cfg, n, nC, size):
    m = meshgen.make_config(cfg, n=n)
    _check_canonical(m)
    assert m.num_clusters == nC and np.all(np.diff(m.cluster_offsets) == size)


def test_config4_variable_clusters():
    m = meshgen.make_config(4, n=32)
    _check_canonical(m)
    sz = np.diff(m.cluster_offsets)
    assert sz.max() <= 2048 and sz.min() >= 1 and sz.max() > 4 * np.median(sz) / 2


def test_deterministic_and_seeded():
    a = meshgen.make_config(3, n=16)
    b = meshgen.make_config(3, n=16)
    assert np.array_equal(a.simplices, b.simplices) and np.array_equal(a.cluster_offsets, b.cluster_offsets)
    c = meshgen.make_mesh(3, 16, clustering="octree", capacity=4096, permute=True, seed=999, keep_fields=True)
    d = meshgen.make_config(3, n=16, keep_fields=True)
    assert not np.array_equal(c.coords, d.coords)


def test_octree_leaves_are_spatial_boxes():
    m = meshgen.make_mesh(3, 16, clustering="octree", capacity=512, seed=4, keep_fields=True)
    assert m.num_clusters == 8
    for c in range(8):
        xyz = m.coords[m.cluster_offsets[c]:m.cluster_offsets[c + 1]]
        ext = xyz.max(0) - xyz.min(0)
        assert np.all(ext < 8.0)                                             # one octant of a 16^3 grid


def test_perforated_is_subset():
    full = meshgen.make_mesh(3, 6, clustering="octree", capacity=30, seed=8)
    holes = meshgen.make_mesh(3, 6, clustering="octree", capacity=30, seed=8, drop_frac=0.15)
    _check_canonical(holes)
    fs = {tuple(r) for r in full.simplices.tolist()}
    assert 0.7 * len(fs) < holes.num_simplices < 0.95 * len(fs)
    assert all(tuple(r) in fs for r in holes.simplices.tolist())
