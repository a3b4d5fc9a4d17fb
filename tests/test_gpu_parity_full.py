"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (batches of 64
clusters, default tile size, device ring, kernel chosen at create): configs 2-5 (config 1 is the small case
of test_gpu_parity.py).

Compared element by element, bit-exactly, with the CPU oracle:
  * config 3 (12.3 M tets): EVERY cluster, against the oracle's global pass (compared fraction 100 %);
  * configs 2, 4, 5: every cluster of one whole batch in every 8 (batches 0, 8, 16, .. and the last one:
    >= 12.5 % of all clusters, spread over the whole mesh), against the oracle's restricted evaluation
    (pinned to the global definitions by tests/test_oracle_pins.py); on config 4, the graded mesh with the
    most diverse tiles, the batches holding the largest cluster, a smallest cluster and the cluster with
    the most simplices whose second vertex leaves the cluster (cross-cluster facets) are added.
Over one complete pass of every cluster, properties that hold at any size — the closed forms of an n^dim
Kuhn/Freudenthal grid (tests/golden/kuhn_closed_forms.txt: 3-D E = 3n^2 m + 3n m^2 + m^3, boundary facets
12 m^2; 2-D E = 2nm + m^2, boundary edges 4m; m = n-1):
        sum |VT| = (dim+1) T,   sum |VV| = 2 E,   #(-1 in TT) = boundary facets,
plus CSR well-formedness of every batch (offsets start at 0, are non-decreasing and end at nnz; indices in
range; every TT entry is -1 or a valid simplex id other than its own row).
Permutation (config 3), coordinate warp (config 4) and clustering change the numbering only, so the
closed forms apply to all four.
"""
import numpy as np
import pytest

import meshgen
import oracle

pytestmark = pytest.mark.gpu

BATCH = 64                       # bench.py --batch default
GRID_N = {2: 4096, 3: 128, 4: 192, 5: 256}   # BASELINE.json configs[1..4]


def _closed_forms(dim, n):
    m = n - 1
    if dim == 3:
        return dict(T=6 * m ** 3, E=3 * n * n * m + 3 * n * m * m + m ** 3, boundary=12 * m * m)
    return dict(T=2 * m * m, E=2 * n * m + m * m, boundary=4 * m)


def _compare(got, ref, what):
    assert len(got) == len(ref)
    for g, r in zip(got, ref):
        c = r["cluster"]
        assert g["cluster"] == c
        for k in ("vt", "vv"):
            assert np.array_equal(g[k][0], r[k][0]), f"{what} {k} offsets, cluster {c}"
            assert np.array_equal(g[k][1], r[k][1]), f"{what} {k} indices, cluster {c}"
        assert g["tt"].shape == r["tt"].shape, f"{what} tt shape, cluster {c}"
        assert np.array_equal(g["tt"], r["tt"]), f"{what} tt, cluster {c}"


@pytest.mark.parametrize("cfg", [2, 3, 4, 5])
def test_full_size_in_bench_configuration(cfg):
    _full_size(cfg, None)


@pytest.mark.parametrize("kernel", ["dense", "walk"])
@pytest.mark.parametrize("cfg", [3, 4])
def test_full_size_with_each_kernel(cfg, kernel):
    """The create-time choice checks one of the two shipped kernels per mesh; here both are forced at full size on the
    permuted grid (config 3) and on the graded one (config 4, the most diverse tiles), same comparison."""
    _full_size(cfg, kernel)


def _full_size(cfg, kernel):
    import torch
    import paper_2507_15230_b200 as gale

    m = meshgen.make_config(cfg)
    D = m.dim + 1
    cf = _closed_forms(m.dim, GRID_N[cfg])
    nT, nV, nC = m.num_simplices, m.num_vertices, m.num_clusters
    assert nT == cf["T"] and nV == GRID_N[cfg] ** m.dim

    gm = gale.GaleMesh(m.dim, nV, m.simplices, m.cluster_offsets, max_batch_clusters=BATCH, queue_depth=0,
                       device_ring=4, tile_vertices=0,                   # exactly bench.py's handle (kernel None)
                       flags={None: 0, "dense": gale.KERNEL_DENSE, "walk": gale.KERNEL_WALK}[kernel])
    if kernel is not None:
        assert gm.info.kernel_variant == (1 if kernel == "walk" else 0)
    assert gm.info.vt_nnz == D * nT                                      # sizes fixed at create
    assert gm.info.vv_nnz == 2 * cf["E"]

    batches = [np.arange(b, min(nC, b + BATCH), dtype=np.int32) for b in range(0, nC, BATCH)]
    first_tet = np.searchsorted(m.simplices[:, 0], m.cluster_offsets)    # I_T per cluster (host, for row ids)
    if cfg == 3:
        sampled_batches = set(range(len(batches)))                      # everything
    else:
        sampled_batches = set(range(0, len(batches), 8)) | {len(batches) - 1}
    if cfg == 4:                                                         # force the extreme clusters in
        sizes = np.diff(m.cluster_offsets)
        second = m.simplices[:, 1]
        owner_hi = m.cluster_offsets[1:][np.searchsorted(m.cluster_offsets, m.simplices[:, 0], side="right") - 1]
        crossing = np.add.reduceat((second >= owner_hi).astype(np.int64), np.minimum(first_tet[:-1], nT - 1))
        crossing[first_tet[1:] == first_tet[:-1]] = 0
        for c in (int(sizes.argmax()), int(sizes.argmin()), int(crossing.argmax())):
            sampled_batches.add(c // BATCH)
    kept = []                                                            # host copies of the compared clusters
    tot = dict(vt=0, vv=0, minus1=0, rows=0, tt_rows=0)

    for bi, ids in enumerate(batches):
        assert gm.compute(ids) == gale.OK
        st, v = gm.pop(-1)
        assert st == gale.OK and v.on_device == 1 and v.n_clusters == len(ids)
        a = gm.view_arrays(v)                                            # torch views of the device slot
        for k in ("vt", "vv"):
            off, idx = a[k + "_offsets"], a[k + "_indices"]
            assert int(off[0]) == 0 and int(off[-1]) == idx.numel()
            assert bool((off[1:] >= off[:-1]).all()), f"{k} offsets not monotone, batch {bi}"
            if idx.numel():
                assert int(idx.min()) >= 0 and int(idx.max()) < (nT if k == "vt" else nV)
            tot[k] += idx.numel()
        tt = a["tt_indices"].view(-1, D)
        t_begin = int(first_tet[ids[0]])
        assert tt.shape[0] == int(first_tet[ids[-1] + 1]) - t_begin      # contiguous cluster ids: one tet range
        own = torch.arange(t_begin, t_begin + tt.shape[0], device=tt.device, dtype=tt.dtype).unsqueeze(1)
        assert bool(((tt >= -1) & (tt < nT) & (tt != own)).all()), f"tt entry out of range, batch {bi}"
        tot["minus1"] += int((tt == -1).sum())
        tot["rows"] += a["vt_offsets"].numel() - 1
        tot["tt_rows"] += tt.shape[0]
        if bi in sampled_batches:
            host = {k: (x.cpu().numpy() if hasattr(x, "cpu") else x) for k, x in a.items()}
            kept += gale.split_batch(host, D)                            # the whole batch
        gm.release(v)

    assert tot["rows"] == nV and tot["tt_rows"] == nT                    # every row exactly once
    assert tot["vt"] == D * nT, "sum |VT| = (dim+1) T"
    assert tot["vv"] == 2 * cf["E"], "sum |VV| = 2 E (closed form)"
    assert tot["minus1"] == cf["boundary"], "#(-1 in TT) = boundary facets (closed form)"
    info = gm.info
    gm.destroy()

    sel = [k["cluster"] for k in kept]
    assert len(sel) >= (nC if cfg == 3 else nC // 8)
    ref = oracle.cluster_results(m.dim, nV, m.simplices, m.cluster_offsets, sel, restricted=(cfg != 3))
    _compare(kept, ref, f"config {cfg} full size (tile {info.tile_vertices}, {info.local_id_bytes}-byte local ids)")


def test_edges_triangles_ve_vf_full_size():
    """SURVEY §8(f)-2 at full size. Config 3 (12.3 M tets): E, F, I_E, I_F and the VE / VF rows of EVERY cluster
    against the oracle's sorted unique combinations. Config 5 (99.5 M tets): the numbers of edges and triangles
    against the Kuhn closed forms (E = 3n^2 m + 3n m^2 + m^3, F = 12 m^3 + 6 m^2), and sum |VE| = 2E,
    sum |VF| = 3F over a complete pass."""
    import paper_2507_15230_b200 as gale
    from test_gpu_sub import gm_array, _rows

    m = meshgen.make_config(3)
    nV, T = m.num_vertices, m.simplices
    gm = gale.GaleMesh(3, nV, T, m.cluster_offsets, max_batch_clusters=BATCH, device_ring=2,
                       flags=gale.WITH_EDGES | gale.WITH_FACETS)
    E = oracle.sub_simplices(3, nV, T, 2)
    F = oracle.sub_simplices(3, nV, T, 3)
    first, upper, nE = gale.gale_mesh_edges(gm.handle)
    ffirst, bc, nF = gale.gale_mesh_triangles(gm.handle)
    assert nE == len(E["list"]) and nF == len(F["list"])
    assert np.array_equal(gm_array(gm, first, nV + 1), E["first"]) and np.array_equal(gm_array(gm, upper, nE), E["list"][:, 1])
    assert np.array_equal(gm_array(gm, ffirst, nV + 1), F["first"])
    assert np.array_equal(gm_array(gm, bc, 2 * nF).reshape(-1, 2), F["list"][:, 1:])
    for b in range(0, m.num_clusters, BATCH):
        ids = list(range(b, min(m.num_clusters, b + BATCH)))
        for g in gale.split_batch(gm.run_batch(ids, gale.REL_VE | gale.REL_VF), 4):
            lo, hi = int(m.cluster_offsets[g["cluster"]]), int(m.cluster_offsets[g["cluster"] + 1])
            off, idx = _rows(E, lo, hi)
            assert np.array_equal(g["ve"][0], off) and np.array_equal(g["ve"][1], idx), f"VE cluster {g['cluster']}"
            off, idx = _rows(F, lo, hi)
            assert np.array_equal(g["vf"][0], off) and np.array_equal(g["vf"][1], idx), f"VF cluster {g['cluster']}"
    gm.destroy()
    del E, F

    m = meshgen.make_config(5)
    n, mm = GRID_N[5], GRID_N[5] - 1
    gm = gale.GaleMesh(3, m.num_vertices, m.simplices, m.cluster_offsets, max_batch_clusters=BATCH, device_ring=2,
                       flags=gale.WITH_EDGES | gale.WITH_FACETS)
    nE_cf, nF_cf = 3 * n * n * mm + 3 * n * mm * mm + mm ** 3, 12 * mm ** 3 + 6 * mm * mm
    assert gm.info.num_edges == nE_cf and gm.info.num_triangles == nF_cf
    tot_ve = tot_vf = 0
    for b in range(0, m.num_clusters, BATCH):
        ids = np.arange(b, min(m.num_clusters, b + BATCH), dtype=np.int32)
        assert gm.compute(ids, gale.REL_VE | gale.REL_VF) == gale.OK
        st, v = gm.pop(-1)
        a = gm.view_arrays(v)
        assert int(a["vf_offsets"][-1]) == a["vf_indices"].numel() and bool((a["vf_offsets"][1:] >= a["vf_offsets"][:-1]).all())
        assert int(a["ve_indices"].max()) < nE_cf and int(a["vf_indices"].max()) < nF_cf and int(a["vf_indices"].min()) >= 0
        tot_ve += a["ve_indices"].numel()
        tot_vf += a["vf_indices"].numel()
        gm.release(v)
    assert tot_ve == 2 * nE_cf and tot_vf == 3 * nF_cf
    gm.destroy()


def test_coboundary_and_boundary_relations_full_size():
    """The rest of SURVEY §8(f)-2 at full size (PAPER.md:309: the relation set of the MS complex; :186-192: the boundary
    look-up). Config 3 (12.3 M tets, 14.5 M edges, 24.7 M triangles):
      * EF / ET / FT of EVERY cluster, element by element against oracle.coboundary (batches of 64, capacities
        rows_cap / star sizes / slot bounds as create derives them at this size);
      * FE / TE / TF of every row against the oracle's sorted lists E and F: entry j of a row must be the id of the row's
        j-th vertex combination in lexicographic order, i.e. list[id] == that combination (ids are unique per
        combination, so this fixes every entry).
    Config 5 (99.5 M tets): the closed forms sum |ET| = 6 T, sum |FT| = 4 T, sum |EF| = 3 F over a complete pass."""
    import itertools

    import paper_2507_15230_b200 as gale

    m = meshgen.make_config(3)
    nV, T, off = m.num_vertices, m.simplices, m.cluster_offsets
    gm = gale.GaleMesh(3, nV, T, off, max_batch_clusters=BATCH, device_ring=2,
                       flags=gale.WITH_EDGES | gale.WITH_FACETS | gale.WITH_COBOUNDARY)
    E = oracle.sub_simplices(3, nV, T, 2)
    F = oracle.sub_simplices(3, nV, T, 3)
    # boundary look-ups, every row
    for rel, rows, lst, width in ((gale.BND_TE, T, E["list"], 2), (gale.BND_TF, T, F["list"], 3), (gale.BND_FE, F["list"], E["list"], 2)):
        got = gm.boundary(rel, 0, len(rows)).cpu().numpy()
        combos = list(itertools.combinations(range(rows.shape[1]), width))
        assert got.shape == (len(rows), len(combos))
        assert got.min() >= 0 and got.max() < len(lst)
        for j, c in enumerate(combos):
            assert np.array_equal(lst[got[:, j]], rows[:, list(c)]), f"boundary relation {rel}, entry {j}"
        del got
    first = {"ef": E["first"], "et": E["first"], "ft": F["first"]}
    for name, bit in (("et", gale.REL_ET), ("ft", gale.REL_FT), ("ef", gale.REL_EF)):   # one oracle relation in memory at a time
        r_off, r_idx = oracle.coboundary(3, nV, T, name.upper())
        for b in range(0, m.num_clusters, BATCH):
            ids = list(range(b, min(m.num_clusters, b + BATCH)))
            for g in gale.split_batch(gm.run_batch(ids, bit), 4):
                c = g["cluster"]
                r0, r1 = int(first[name][off[c]]), int(first[name][off[c + 1]])
                o = r_off[r0:r1 + 1]
                assert np.array_equal(g[name][0], (o - o[0]).astype(np.int32)), f"{name} offsets of cluster {c}"
                assert np.array_equal(g[name][1], r_idx[o[0]:o[-1]]), f"{name} of cluster {c}"
        del r_off, r_idx
    gm.destroy()
    del E, F, m, T

    m = meshgen.make_config(5)
    mm = GRID_N[5] - 1
    nT, nF_cf = 6 * mm ** 3, 12 * mm ** 3 + 6 * mm * mm
    gm = gale.GaleMesh(3, m.num_vertices, m.simplices, m.cluster_offsets, max_batch_clusters=BATCH, device_ring=2,
                       flags=gale.WITH_EDGES | gale.WITH_FACETS | gale.WITH_COBOUNDARY)
    assert gm.info.num_triangles == nF_cf
    tot = dict(et=0, ft=0, ef=0)
    for b in range(0, m.num_clusters, BATCH):
        ids = np.arange(b, min(m.num_clusters, b + BATCH), dtype=np.int32)
        assert gm.compute(ids, gale.REL_ET | gale.REL_FT | gale.REL_EF) == gale.OK
        st, v = gm.pop(-1)
        assert st == gale.OK
        tot["et"] += int(v.et_nnz); tot["ft"] += int(v.ft_nnz); tot["ef"] += int(v.ef_nnz)
        a = gm.view_arrays(v)
        for k in ("et", "ft", "ef"):
            o = a[k + "_offsets"]
            assert int(o[0]) == 0 and int(o[-1]) == a[k + "_indices"].numel() == int(getattr(v, k + "_nnz"))
            assert bool((o[1:] > o[:-1]).all())                       # every edge / triangle has a coface
        assert int(a["ft_indices"].max()) < nT and int(a["ef_indices"].max()) < nF_cf
        gm.release(v)
    assert tot["et"] == 6 * nT and tot["ft"] == 4 * nT and tot["ef"] == 3 * nF_cf
    gm.destroy()
