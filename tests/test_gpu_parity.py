"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
bit-exact (integer index work), on the same seeded meshes."""
import numpy as np
import pytest

import meshgen
import oracle

pytestmark = pytest.mark.gpu


def _gale():
    import paper_2507_15230_b200 as gale
    return gale


def _compare(got, ref, what=""):
    assert len(got) == len(ref)
    for g, r in zip(got, ref):
        c = r["cluster"]
        assert g["cluster"] == c
        for k in ("vt", "vv"):
            if k in g:
                assert np.array_equal(g[k][0], r[k][0]), f"{what} {k} offsets, cluster {c}"
                assert np.array_equal(g[k][1], r[k][1]), f"{what} {k} indices, cluster {c}"
        if "tt" in g:
            assert g["tt"].shape == r["tt"].shape, f"{what} tt shape, cluster {c}"
            bad = np.nonzero(g["tt"] != r["tt"])
            assert len(bad[0]) == 0, f"{what} tt, cluster {c}: first diff row {bad[0][:3]} col {bad[1][:3]}"


def _run_all(m, batch, restricted=False, clusters=None, **kw):
    gale = _gale()
    gm = gale.GaleMesh(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, max_batch_clusters=batch, **kw)
    ids = list(range(m.num_clusters)) if clusters is None else list(clusters)
    got = []
    for b in range(0, len(ids), batch):
        got += gale.split_batch(gm.run_batch(ids[b:b + batch]), m.dim + 1)
    ref = oracle.cluster_results(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, ids, restricted=restricted)
    info = gm.info
    gm.destroy()
    return got, ref, info


SMALL = [
    ("cfg1", lambda: meshgen.make_config(1), 8),
    ("cfg2@256", lambda: meshgen.make_config(2, n=256), 5),
    ("cfg3@40", lambda: meshgen.make_config(3, n=40), 7),
    ("cfg4@40", lambda: meshgen.make_config(4, n=40), 64),
    ("cfg5@48", lambda: meshgen.make_config(5, n=48), 64),
    ("holes3d", lambda: meshgen.make_mesh(3, 24, clustering="octree", capacity=700, permute=True, drop_frac=0.15, seed=5), 16),
    ("holes2d", lambda: meshgen.make_mesh(2, 150, clustering="octree", capacity=900, warp=True, drop_frac=0.2, seed=6), 16),
    # irregular meshes (Delaunay of random points: |VT| up to ~60 against a mean of 26)
    ("delaunay3d", lambda: meshgen.make_delaunay(3, 6000, seed=31, capacity=600), 8),
    ("delaunay2d", lambda: meshgen.make_delaunay(2, 20000, seed=32, capacity=1500), 8),
]


KERNELS = {"auto": 0, "dense": 8, "walk": 16}       # GALE_KERNEL_DENSE / GALE_KERNEL_WALK; auto = timed choice at create


def _run_kernel(m, batch, kernel, **kw):
    """_run_all with a forced kernel variant; skips when the walk kernel's capacity limits refuse the mesh."""
    gale = _gale()
    flags = kw.pop("flags", gale.VALIDATE) | KERNELS[kernel]
    try:
        got, ref, info = _run_all(m, batch, flags=flags, **kw)
    except gale.GaleError as e:
        if kernel == "walk" and e.status == gale.ERR_UNSUPPORTED:
            pytest.skip("walk kernel does not admit this mesh")
        raise
    if kernel != "auto":
        assert info.kernel_variant == (1 if kernel == "walk" else 0)
    return got, ref, info


@pytest.mark.parametrize("kernel", list(KERNELS))
@pytest.mark.parametrize("name,make,batch", SMALL, ids=[s[0] for s in SMALL])
def test_parity_small(name, make, batch, kernel):
    m = make()
    got, ref, _ = _run_kernel(m, batch, kernel)
    _compare(got, ref, f"{name} [{kernel}]")


@pytest.mark.parametrize("kernel", ["dense", "walk"])
@pytest.mark.parametrize("tv", [3, 16, 64])
def test_parity_irregular_mesh_tile_sizes(tv, kernel):
    m = meshgen.make_delaunay(3, 2500, seed=33, capacity=400)
    got, ref, _ = _run_kernel(m, 5, kernel, tile_vertices=tv, flags=3)          # VALIDATE | VALIDATE_MANIFOLD
    _compare(got, ref, f"delaunay3d tv={tv} [{kernel}]")


@pytest.mark.parametrize("kernel", ["dense", "walk"])
@pytest.mark.parametrize("tv", [1, 7, 32, 100, 256])
def test_parity_tile_sizes(tv, kernel):
    """Ragged tiles, one-vertex tiles, and tiles as large as a block."""
    m = meshgen.make_mesh(3, 14, clustering="octree", capacity=300, permute=True, drop_frac=0.1, seed=13)
    got, ref, info = _run_kernel(m, 9, kernel, tile_vertices=tv)
    assert info.tile_vertices <= max(tv, 1)
    _compare(got, ref, f"tv={tv} [{kernel}]")
    m2 = meshgen.make_mesh(2, 60, clustering="octree", capacity=500, seed=14)
    got, ref, _ = _run_kernel(m2, 4, kernel, tile_vertices=tv)
    _compare(got, ref, f"2d tv={tv} [{kernel}]")


def test_both_local_id_widths():
    """The staged lists use 8-bit tile-local vertex ids when every tile has at most 255 local vertices
    and 16-bit ids otherwise; both encodings must be exercised and both must be bit-exact."""
    m = meshgen.make_mesh(3, 20, clustering="octree", capacity=2000, permute=True, drop_frac=0.05, seed=21)
    assert int(np.diff(m.cluster_offsets).max()) >= 256
    got, ref, info = _run_all(m, 4, tile_vertices=16)
    assert info.local_id_bytes == 1
    _compare(got, ref, "8-bit local ids")
    got, ref, info = _run_all(m, 4, tile_vertices=256)
    # tets keep 9-bit local ids in the facet key (<= 512 per tile), so create may halve the requested tile;
    # 128 rows plus their halo still exceed 255 local ids
    assert info.tile_vertices in (128, 256) and info.local_id_bytes == 2
    _compare(got, ref, "16-bit local ids")
    m2 = meshgen.make_mesh(2, 120, clustering="octree", capacity=3000, seed=22)
    for tv, lb in ((32, 1), (256, 2)):
        got, ref, info = _run_all(m2, 3, tile_vertices=tv)
        assert info.local_id_bytes == lb
        _compare(got, ref, f"2d local id bytes {lb}")


@pytest.mark.parametrize("kernel", ["dense", "walk"])
@pytest.mark.parametrize("mask", [1, 2, 4, 3, 5, 6])
def test_relation_masks(mask, kernel):
    gale = _gale()
    m = meshgen.make_config(1)
    gm = gale.GaleMesh(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, max_batch_clusters=8,
                       flags=gale.VALIDATE | KERNELS[kernel])
    host = gm.run_batch([5, 0, 3], mask)
    got = gale.split_batch(host, 4)
    ref = oracle.cluster_results(3, m.num_vertices, m.simplices, m.cluster_offsets, [5, 0, 3], mask=mask)
    for g in got:
        assert ("vt" in g) == bool(mask & 1) and ("vv" in g) == bool(mask & 2) and ("tt" in g) == bool(mask & 4)
    _compare(got, ref, f"mask={mask}")
    gm.destroy()


def test_edge_cases_empty_duplicates_order():
    gale = _gale()
    # empty clusters (zero vertices), a cluster with vertices but no internal simplex, isolated vertices
    T = np.array([[0, 1, 2, 3], [1, 2, 3, 9]], np.int32)
    off = np.array([0, 0, 4, 4, 8, 12, 12], np.int32)            # clusters 0,2,5 empty; cluster 3 = {4..7} isolated
    gm = gale.GaleMesh(3, 12, T, off, max_batch_clusters=8)
    ids = [4, 1, 1, 0, 3, 5, 2]                                   # duplicates legal, order kept
    got = gale.split_batch(gm.run_batch(ids), 4)
    ref = oracle.cluster_results(3, 12, T, off, ids)
    _compare(got, ref, "edge")
    # an empty batch is legal and yields empty CSR
    host = gm.run_batch([])
    assert host["n_clusters"] == 0 and host["vt_offsets"].tolist() == [0] and host["vv_offsets"].tolist() == [0]
    assert host["tt_indices"].size == 0
    gm.destroy()
    # a mesh without simplices
    gm = gale.GaleMesh(2, 6, np.zeros((0, 3), np.int32), np.array([0, 3, 6], np.int32), max_batch_clusters=2)
    host = gm.run_batch([1, 0])
    assert host["vt_offsets"].tolist() == [0] * 7 and host["vv_indices"].size == 0 and host["tt_indices"].size == 0
    gm.destroy()


def test_fig1_toy_on_gpu():
    gale = _gale()
    m = meshgen.toy_two_tets()
    gm = gale.GaleMesh(3, 5, m.simplices, m.cluster_offsets, max_batch_clusters=1)
    g = gale.split_batch(gm.run_batch([0]), 4)[0]
    assert g["vv"][1][g["vv"][0][0]:g["vv"][0][1]].tolist() == [1, 2, 3]
    assert g["tt"].tolist() == [[1, -1, -1, -1], [-1, -1, -1, 0]]
    gm.destroy()


def test_determinism_same_batch_twice():
    gale = _gale()
    m = meshgen.make_config(3, n=32)
    gm = gale.GaleMesh(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, max_batch_clusters=8)
    a = gm.run_batch(list(range(8)))
    b = gm.run_batch(list(range(8)))
    for k in ("vt_offsets", "vt_indices", "vv_offsets", "vv_indices", "tt_indices"):
        assert np.array_equal(a[k], b[k]), k
    gm.destroy()


def test_queue_protocol_pinned_and_device():
    gale = _gale()
    m = meshgen.make_config(1)
    ref = oracle.cluster_results(3, m.num_vertices, m.simplices, m.cluster_offsets, range(8))
    for depth, ring in ((2, 0), (0, 3)):
        gm = gale.GaleMesh(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, max_batch_clusters=2,
                           queue_depth=depth, device_ring=ring)
        nslots = depth or ring
        st, _ = gm.pop(0)
        assert st == gale.ERR_EMPTY
        for i in range(nslots):
            assert gm.compute([2 * i, 2 * i + 1]) == gale.OK
        assert gm.compute([0, 1]) == gale.ERR_WOULD_BLOCK          # bounded queue: back-pressure
        views = []
        for i in range(nslots):                                    # FIFO
            st, v = gm.pop(-1)
            assert st == gale.OK and v.sequence == i and v.on_device == (1 if depth == 0 else 0)
            arr = gm.view_arrays(v)
            host = {k: (x.cpu().numpy() if hasattr(x, "cpu") else x) for k, x in arr.items()}
            _compare(gale.split_batch(host, 4), ref[2 * i:2 * i + 2], f"queue depth={depth}")
            views.append(v)
        assert gm.compute([0, 1]) == gale.ERR_WOULD_BLOCK          # popped but not released
        gm.release(views[0])
        assert gm.compute([6, 7]) == gale.OK
        st, v = gm.pop(-1)
        assert st == gale.OK and v.sequence == nslots
        gm.release(v)
        for v in views[1:]:
            gm.release(v)
        with pytest.raises(gale.GaleError):
            gm.release(views[0])                                   # double release
        gm.destroy()


def test_argument_errors_on_gpu():
    gale = _gale()
    m = meshgen.make_config(1)
    gm = gale.GaleMesh(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, max_batch_clusters=4)
    for ids, mask, status in (([0, 8], 7, gale.ERR_BAD_CLUSTER), ([-1], 7, gale.ERR_BAD_CLUSTER),
                              ([0, 1, 2, 3, 4], 7, gale.ERR_BAD_CLUSTER), ([0], 0, gale.ERR_INVALID_ARG),
                              ([0], 1 << 20, gale.ERR_INVALID_ARG),                          # not a relation bit
                              ([0], gale.REL_VE, gale.ERR_UNSUPPORTED), ([0], gale.REL_EF, gale.ERR_UNSUPPORTED)):  # lists not built
        with pytest.raises(gale.GaleError) as e:
            gm.compute(ids, mask)
        assert e.value.status == status
    gm.destroy()
    T = m.simplices.copy()
    T[[10, 11]] = T[[11, 10]]
    with pytest.raises(gale.GaleError) as e:
        gale.GaleMesh(3, m.num_vertices, T, m.cluster_offsets)
    assert e.value.status == gale.ERR_NOT_CANONICAL
    tri = np.array([[0, 1, 2], [0, 1, 3], [0, 1, 4]], np.int32)
    with pytest.raises(gale.GaleError) as e:
        gale.GaleMesh(2, 5, tri, np.array([0, 5], np.int32), flags=gale.VALIDATE | gale.VALIDATE_MANIFOLD)
    assert e.value.status == gale.ERR_NONMANIFOLD


def test_large_batch_splits_launches():
    """More clusters than one kernel-parameter descriptor holds (128): several launches, one slot."""
    m = meshgen.make_config(4, n=40)
    assert m.num_clusters > 128
    got, ref, _ = _run_all(m, m.num_clusters)
    _compare(got, ref, "big batch")


@pytest.mark.parametrize("name,make,batch", SMALL[:5] + SMALL[7:8], ids=[s[0] for s in SMALL[:5] + SMALL[7:8]])
def test_parity_staging_from_t(name, make, batch):
    """Dense kernel with GALE_STAGE_FROM_T: the rows of T and T_ex are staged and mapped to tile-local ids in
    the kernel (SURVEY §8 a1 as written) instead of reading the create-time re-encoding."""
    gale = _gale()
    m = make()
    got, ref, info = _run_all(m, batch, flags=gale.VALIDATE | gale.KERNEL_DENSE | gale.STAGE_FROM_T)
    assert info.kernel_variant == 0
    _compare(got, ref, f"{name} [stage from T]")


def test_staging_from_t_selects_the_dense_kernel():
    """GALE_STAGE_FROM_T alone (no GALE_KERNEL_DENSE): the flag must not become a silent no-op when the create-time
    timing would have picked the walk kernel (which cannot stage from T)."""
    gale = _gale()
    m = meshgen.make_config(1)                      # a regular grid: the walk kernel's home ground
    got, ref, info = _run_all(m, 8, flags=gale.VALIDATE | gale.STAGE_FROM_T)
    assert info.kernel_variant == 0 and info.tune_walk_ms == 0.0
    _compare(got, ref, "cfg1 [stage from T, kernel not named]")
