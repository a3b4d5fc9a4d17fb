"""Edges / triangles and the coboundary relations VE / VF (Table 1) through the
C ABI against the CPU oracle (oracle.sub_simplices: sorted unique combinations, plain definitions), bit-exact:
the lists E and F with their interval arrays as the initialization builds them on the device, and the VE / VF
rows of cluster batches."""
import numpy as np
import pytest

import meshgen
import oracle

pytestmark = pytest.mark.gpu

CASES = [
    ("cfg1", lambda: meshgen.make_config(1), 8, 3),
    ("cfg3@32", lambda: meshgen.make_config(3, n=32), 5, 3),
    ("holes3d", lambda: meshgen.make_mesh(3, 20, clustering="octree", capacity=500, permute=True, drop_frac=0.15, seed=5), 7, 3),
    ("delaunay3d", lambda: meshgen.make_delaunay(3, 4000, seed=31, capacity=500), 4, 3),
    ("tri2d (VE only)", lambda: meshgen.make_mesh(2, 80, clustering="octree", capacity=700, drop_frac=0.1, seed=6), 5, 2),
]


def _rows(s, lo, hi):
    off = s["v_off"][lo:hi + 1]
    return (off - off[0]).astype(np.int32), s["v_idx"][off[0]:off[-1]]


@pytest.mark.parametrize("kernel", ["dense", "walk"])
@pytest.mark.parametrize("name,make,batch,dim", CASES, ids=[c[0] for c in CASES])
def test_edges_triangles_ve_vf(name, make, batch, dim, kernel):
    import paper_2507_15230_b200 as gale

    m = make()
    assert m.dim == dim
    T, nV = m.simplices, m.num_vertices
    flags = gale.VALIDATE | gale.WITH_EDGES | (gale.WITH_FACETS if dim == 3 else 0)
    flags |= gale.KERNEL_WALK if kernel == "walk" else gale.KERNEL_DENSE
    try:
        gm = gale.GaleMesh(dim, nV, T, m.cluster_offsets, max_batch_clusters=batch, flags=flags)
    except gale.GaleError as e:
        if kernel == "walk" and e.status == gale.ERR_UNSUPPORTED:
            pytest.skip("walk kernel does not admit this mesh")
        raise
    E = oracle.sub_simplices(dim, nV, T, 2)
    # the edge list and its interval array as built on the device
    first, upper, nE = gale.gale_mesh_edges(gm.handle)
    assert nE == len(E["list"]) == gm.info.num_edges
    e_first = gm_array(gm, first, nV + 1)
    assert np.array_equal(e_first, E["first"])
    assert np.array_equal(gm_array(gm, upper, nE), E["list"][:, 1])
    assert np.array_equal(np.repeat(np.arange(nV), np.diff(e_first)), E["list"][:, 0])
    mask = gale.REL_VE
    if dim == 3:
        F = oracle.sub_simplices(dim, nV, T, 3)
        ffirst, bc, nF = gale.gale_mesh_triangles(gm.handle)
        assert nF == len(F["list"]) == gm.info.num_triangles
        assert np.array_equal(gm_array(gm, ffirst, nV + 1), F["first"])
        assert np.array_equal(gm_array(gm, bc, 2 * nF).reshape(-1, 2), F["list"][:, 1:])
        mask |= gale.REL_VF
    ids = list(range(m.num_clusters))[::-1]                         # any order, several batches
    ref = oracle.cluster_results(dim, nV, T, m.cluster_offsets, ids, mask=3)
    k = 0
    for b in range(0, len(ids), batch):
        host = gm.run_batch(ids[b:b + batch], mask)
        assert host["relation_mask"] & gale.REL_VV                  # VE delivers VV too
        for g in gale.split_batch(host, dim + 1):
            c = g["cluster"]
            lo, hi = int(m.cluster_offsets[c]), int(m.cluster_offsets[c + 1])
            assert np.array_equal(g["vv"][1], ref[k]["vv"][1])
            off, idx = _rows(E, lo, hi)
            assert np.array_equal(g["ve"][0], off) and np.array_equal(g["ve"][1], idx), f"{name}: VE of cluster {c}"
            if dim == 3:
                off, idx = _rows(F, lo, hi)
                assert np.array_equal(g["vf"][0], off), f"{name}: VF offsets of cluster {c}"
                assert np.array_equal(g["vf"][1], idx), f"{name}: VF of cluster {c}"
                assert "vt" not in g                                # VF is read off the VV rows, like VE
            k += 1
    # all five relations in one call
    if dim == 3:
        host = gm.run_batch(ids[:batch], gale.REL_ALL | gale.REL_VE | gale.REL_VF)
        full = oracle.cluster_results(dim, nV, T, m.cluster_offsets, ids[:batch])
        for g, r in zip(gale.split_batch(host, dim + 1), full):
            assert np.array_equal(g["tt"], r["tt"]) and np.array_equal(g["vv"][1], r["vv"][1])
            lo, hi = int(m.cluster_offsets[g["cluster"]]), int(m.cluster_offsets[g["cluster"] + 1])
            assert np.array_equal(g["vf"][1], _rows(F, lo, hi)[1]) and np.array_equal(g["ve"][1], _rows(E, lo, hi)[1])
    gm.destroy()


def gm_array(gm, ptr, n):
    """int32 host copy of n entries at a DEVICE address owned by the library (not inside the caller's workspace)."""
    from cuda.bindings import runtime as cudart

    out = np.empty(max(n, 1), np.int32)
    if n:
        (err,) = cudart.cudaMemcpy(out.ctypes.data, ptr, 4 * n, cudart.cudaMemcpyKind.cudaMemcpyDeviceToHost)
        assert int(err) == 0, err
    return out[:n]


def test_ve_vf_need_the_lists():
    import paper_2507_15230_b200 as gale

    m = meshgen.make_config(1)
    gm = gale.GaleMesh(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, max_batch_clusters=4)
    for mask in (gale.REL_VE, gale.REL_VF):
        with pytest.raises(gale.GaleError) as e:
            gm.compute([0], mask)
        assert e.value.status == gale.ERR_UNSUPPORTED
    gm.destroy()
    tri = meshgen.make_mesh(2, 20, clustering="octree", capacity=100, seed=3)
    with pytest.raises(gale.GaleError) as e:
        gale.GaleMesh(2, tri.num_vertices, tri.simplices, tri.cluster_offsets, flags=gale.WITH_FACETS)
    assert e.value.status == gale.ERR_INVALID_ARG


COB_CASES = [
    ("cfg1", lambda: meshgen.make_config(1), 8),
    ("cfg3@32", lambda: meshgen.make_config(3, n=32), 5),
    ("holes3d", lambda: meshgen.make_mesh(3, 20, clustering="octree", capacity=500, permute=True, drop_frac=0.15, seed=5), 7),
    ("delaunay3d", lambda: meshgen.make_delaunay(3, 4000, seed=31, capacity=500), 4),
]


@pytest.mark.parametrize("name,make,batch", COB_CASES, ids=[c[0] for c in COB_CASES])
def test_ef_et_ft(name, make, batch):
    """EF / ET / FT of cluster batches (rows = the clusters' own edges / triangles) against the oracle's plain
    coboundary definition, bit-exact; several batches, clusters in reverse order, and all eight relations at once."""
    import paper_2507_15230_b200 as gale

    m = make()
    T, nV = m.simplices, m.num_vertices
    gm = gale.GaleMesh(3, nV, T, m.cluster_offsets, max_batch_clusters=batch, device_ring=2,
                       flags=gale.VALIDATE | gale.WITH_EDGES | gale.WITH_FACETS | gale.WITH_COBOUNDARY)
    E = oracle.sub_simplices(3, nV, T, 2)
    F = oracle.sub_simplices(3, nV, T, 3)
    ref = {k: oracle.coboundary(3, nV, T, k.upper()) for k in ("ef", "et", "ft")}
    first = {"ef": E["first"], "et": E["first"], "ft": F["first"]}
    ids = list(range(m.num_clusters))[::-1]
    mask = gale.REL_EF | gale.REL_ET | gale.REL_FT
    for b in range(0, len(ids), batch):
        if b == 0:
            host = gm.run_batch(ids[b:b + batch], mask | gale.REL_ALL | gale.REL_VE | gale.REL_VF)
        else:
            host = gm.run_batch(ids[b:b + batch], mask)
        for g in gale.split_batch(host, 4):
            c = g["cluster"]
            lo, hi = int(m.cluster_offsets[c]), int(m.cluster_offsets[c + 1])
            for k in ("ef", "et", "ft"):
                r0, r1 = int(first[k][lo]), int(first[k][hi])
                off = ref[k][0][r0:r1 + 1]
                assert np.array_equal(g[k][0], (off - off[0]).astype(np.int32)), f"{name}: {k} offsets of cluster {c}"
                assert np.array_equal(g[k][1], ref[k][1][off[0]:off[-1]]), f"{name}: {k} of cluster {c}"
            if b == 0:
                assert "tt" in g and "ve" in g and "vf" in g
    gm.destroy()


@pytest.mark.parametrize("kernel", ["dense", "walk"])
def test_batches_larger_than_one_launch(kernel):
    """A batch of 200 clusters is split over two kernel launches (128 clusters per batch descriptor, gale_lib.cu):
    the per-launch row / nnz bases of every relation (VT / VV / TT, VE, VF, EF / ET / FT) must continue where the
    previous launch stopped. 587 small clusters, one of them empty, duplicated ids in the batch, all eight relations
    at once, three batches (200 + 200 + a ragged one), against the oracle."""
    import paper_2507_15230_b200 as gale

    m = meshgen.make_mesh(3, 18, clustering="octree", capacity=16, permute=True, drop_frac=0.1, seed=9)
    T, nV = m.simplices, m.num_vertices
    off = np.asarray(m.cluster_offsets)
    off = np.insert(off, 100, off[100]).astype(np.int32)            # cluster 100 owns no vertex
    nC = len(off) - 1
    assert nC > 260 and off[100] == off[101]
    batch = 200
    flags = gale.VALIDATE | gale.WITH_EDGES | gale.WITH_FACETS | gale.WITH_COBOUNDARY
    flags |= gale.KERNEL_WALK if kernel == "walk" else gale.KERNEL_DENSE
    try:
        gm = gale.GaleMesh(3, nV, T, off, max_batch_clusters=batch, device_ring=2, flags=flags)
    except gale.GaleError as e:
        if kernel == "walk" and e.status == gale.ERR_UNSUPPORTED:
            pytest.skip("walk kernel does not admit this mesh")
        raise
    assert gm.info.kernel_variant == (1 if kernel == "walk" else 0)
    rng = np.random.default_rng(4)
    ids = [int(c) for c in rng.permutation(nC)]
    ids[10] = ids[150] = 100                                         # the empty cluster, in both launches of batch 0
    ids[140] = ids[3]                                                # a duplicate across the launch boundary
    ids[199] = ids[198]                                              # and inside the second launch
    E = oracle.sub_simplices(3, nV, T, 2)
    F = oracle.sub_simplices(3, nV, T, 3)
    cob = {k: oracle.coboundary(3, nV, T, k.upper()) for k in ("ef", "et", "ft")}
    first = {"ef": E["first"], "et": E["first"], "ft": F["first"]}
    mask = gale.REL_ALL | gale.REL_VE | gale.REL_VF | gale.REL_EF | gale.REL_ET | gale.REL_FT
    for b in range(0, len(ids), batch):
        chunk = ids[b:b + batch]
        ref = oracle.cluster_results(3, nV, T, off, chunk)
        got = gale.split_batch(gm.run_batch(chunk, mask), 4)
        assert [g["cluster"] for g in got] == chunk
        for g, r in zip(got, ref):
            c = g["cluster"]
            lo, hi = int(off[c]), int(off[c + 1])
            for k in ("vt", "vv"):
                assert np.array_equal(g[k][0], r[k][0]) and np.array_equal(g[k][1], r[k][1]), f"{k} of cluster {c}"
            assert np.array_equal(g["tt"], r["tt"]), f"tt of cluster {c}"
            o, i = _rows(E, lo, hi)
            assert np.array_equal(g["ve"][0], o) and np.array_equal(g["ve"][1], i), f"ve of cluster {c}"
            o, i = _rows(F, lo, hi)
            assert np.array_equal(g["vf"][0], o) and np.array_equal(g["vf"][1], i), f"vf of cluster {c}"
            for k in ("ef", "et", "ft"):
                r0, r1 = int(first[k][lo]), int(first[k][hi])
                o = cob[k][0][r0:r1 + 1]
                assert np.array_equal(g[k][0], (o - o[0]).astype(np.int32)), f"{k} offsets of cluster {c}"
                assert np.array_equal(g[k][1], cob[k][1][o[0]:o[-1]]), f"{k} of cluster {c}"
    gm.destroy()


BND_CASES = [
    ("cfg1", lambda: meshgen.make_config(1)),
    ("holes3d", lambda: meshgen.make_mesh(3, 12, clustering="octree", capacity=200, permute=True, drop_frac=0.15, seed=8)),
    ("delaunay3d", lambda: meshgen.make_delaunay(3, 1500, seed=41, capacity=300)),
]


@pytest.mark.parametrize("name,make", BND_CASES, ids=[c[0] for c in BND_CASES])
def test_boundary_relations_fe_te_tf(name, make):
    """FE / TE / TF by the interval-bounded look-up on the device against the oracle's dictionary
    look-up in the whole list, every row, plus a ragged sub-range."""
    import paper_2507_15230_b200 as gale

    m = make()
    gm = gale.GaleMesh(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, max_batch_clusters=4,
                       flags=gale.WITH_EDGES | gale.WITH_FACETS)
    nF = len(oracle.sub_simplices(3, m.num_vertices, m.simplices, 3)["list"])
    for rel, key, rows in ((gale.BND_FE, "FE", nF), (gale.BND_TE, "TE", len(m.simplices)), (gale.BND_TF, "TF", len(m.simplices))):
        ref = oracle.boundary(3, m.num_vertices, m.simplices, key)
        got = gm.boundary(rel, 0, rows).cpu().numpy()
        assert np.array_equal(got, ref), f"{name}: {key}"
        lo, n = rows // 3 + 1, min(777, rows - rows // 3 - 1)
        assert np.array_equal(gm.boundary(rel, lo, n).cpu().numpy(), ref[lo:lo + n])
        assert gm.boundary(rel, rows, 0).shape[0] == 0
        with pytest.raises(gale.GaleError) as e:
            gm.boundary(rel, rows - 1, 2)
        assert e.value.status == gale.ERR_INVALID_ARG
    gm.destroy()


def test_boundary_te_2d_and_missing_lists():
    import paper_2507_15230_b200 as gale

    tri = meshgen.make_mesh(2, 30, clustering="octree", capacity=150, drop_frac=0.1, seed=3)
    gm = gale.GaleMesh(2, tri.num_vertices, tri.simplices, tri.cluster_offsets, max_batch_clusters=4, flags=gale.WITH_EDGES)
    ref = oracle.boundary(2, tri.num_vertices, tri.simplices, "TE")
    assert np.array_equal(gm.boundary(gale.BND_TE, 0, len(tri.simplices)).cpu().numpy(), ref)
    for rel in (gale.BND_FE, gale.BND_TF):
        with pytest.raises(gale.GaleError) as e:
            gm.boundary(rel, 0, 1)
        assert e.value.status == gale.ERR_UNSUPPORTED
    with pytest.raises(gale.GaleError) as e:
        gm.boundary(7, 0, 1)
    assert e.value.status == gale.ERR_INVALID_ARG
    gm.destroy()
