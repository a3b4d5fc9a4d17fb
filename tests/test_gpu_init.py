"""GPU-side initialization: the interval array I_T and the external
lists T_ex the device kernels build, against the CPU oracle's plain scans (oracle.internal_range /
oracle.external_list, pinned on the paper's Fig. 4 facts), tile by tile; and the tile-local vertex table
against numpy set arithmetic on the staged simplices."""
import numpy as np
import pytest

import meshgen
import oracle

pytestmark = pytest.mark.gpu

CASES = [
    ("cfg1", lambda: meshgen.make_config(1), 0),
    ("cfg3@24 tv=7", lambda: meshgen.make_config(3, n=24), 7),
    ("holes3d", lambda: meshgen.make_mesh(3, 16, clustering="octree", capacity=300, permute=True, drop_frac=0.15, seed=5), 16),
    ("holes2d", lambda: meshgen.make_mesh(2, 60, clustering="octree", capacity=400, warp=True, drop_frac=0.2, seed=6), 0),
    ("delaunay3d", lambda: meshgen.make_delaunay(3, 2500, seed=33, capacity=400), 0),
]


@pytest.mark.parametrize("name,make,tv", CASES, ids=[c[0] for c in CASES])
def test_device_interval_array_and_external_lists(name, make, tv):
    import paper_2507_15230_b200 as gale

    m = make()
    T = m.simplices
    gm = gale.GaleMesh(m.dim, m.num_vertices, T, m.cluster_offsets, max_batch_clusters=4, tile_vertices=tv)
    # I_T per vertex: entry v = number of simplices whose lowest vertex is below v (oracle: plain scan per vertex range)
    first = gm.device_array(gale.gale_mesh_interval_array(gm.handle), m.num_vertices + 1).cpu().numpy()
    assert first[0] == 0 and first[-1] == len(T)
    seen_rows = 0
    for i in range(gm.info.num_tiles):
        v = gale.gale_mesh_tile(gm.handle, i)
        lo, hi = v.v_lo, v.v_lo + v.nrows
        assert m.cluster_offsets[v.cluster] <= lo and hi <= m.cluster_offsets[v.cluster + 1]
        a, b = oracle.internal_range(m.dim, T, lo, hi)
        assert (v.t_lo, v.t_lo + v.num_internal) == (a, b), f"{name}: I_T of tile {i}"
        assert (first[lo], first[hi]) == (a, b)
        ext = gm.device_array(v.d_external, v.num_external).cpu().numpy()
        ref = oracle.external_list(m.dim, T, lo, hi)
        assert np.array_equal(ext, ref), f"{name}: T_ex of tile {i}"
        # local -> global table: [halo below][tile][halo above], ascending
        staged = np.concatenate([T[ref], T[a:b]]) if len(ref) + (b - a) else np.zeros((0, m.dim + 1), np.int32)
        verts = np.unique(staged)
        halo = verts[(verts < lo) | (verts >= hi)]
        want = np.concatenate([halo[halo < lo], np.arange(lo, hi), halo[halo >= hi]]).astype(np.int32)
        got = gm.device_array(v.d_local_to_global, v.num_local).cpu().numpy()
        assert np.array_equal(got, want), f"{name}: vertex table of tile {i}"
        assert v.num_lower_halo == int((halo < lo).sum())
        seen_rows += v.nrows
    assert seen_rows == m.num_vertices
    gm.destroy()


def test_two_handles_with_different_shared_memory_needs():
    """The dynamic shared-memory ceiling belongs to the kernel, not to a handle: a second,
    smaller mesh on the same kernel instantiation must not break launches of the first."""
    import paper_2507_15230_b200 as gale

    big = meshgen.make_delaunay(3, 4000, seed=41, capacity=500)
    small = meshgen.make_config(1)
    for flags in (gale.VALIDATE | gale.KERNEL_DENSE, gale.VALIDATE | gale.KERNEL_WALK):
        g1 = gale.GaleMesh(big.dim, big.num_vertices, big.simplices, big.cluster_offsets, max_batch_clusters=4, flags=flags)
        g2 = gale.GaleMesh(small.dim, small.num_vertices, small.simplices, small.cluster_offsets, max_batch_clusters=4, flags=flags)
        assert g1.info.smem_bytes != g2.info.smem_bytes
        for g, mm in ((g1, big), (g2, small), (g1, big)):
            got = gale.split_batch(g.run_batch([0, 1]), mm.dim + 1)
            ref = oracle.cluster_results(mm.dim, mm.num_vertices, mm.simplices, mm.cluster_offsets, [0, 1])
            for a, r in zip(got, ref):
                assert np.array_equal(a["vt"][1], r["vt"][1]) and np.array_equal(a["vv"][1], r["vv"][1])
                assert np.array_equal(a["tt"], r["tt"])
        g1.destroy()
        g2.destroy()


def test_stream_ordered_flag():
    """GALE_STREAM_ORDERED: the batch kernels run on the caller's stream, so work enqueued on that stream
    afterwards sees the finished device slot without gale_queue_pop having synchronised anything."""
    import torch
    import paper_2507_15230_b200 as gale

    m = meshgen.make_config(3, n=32)
    gm = gale.GaleMesh(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, max_batch_clusters=8,
                       flags=gale.VALIDATE | gale.STREAM_ORDERED)
    ids = list(range(8))
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        assert gm.compute(ids, stream=st) == gale.OK
        # a copy enqueued on the same stream right after the batch: ordered after the kernels by the stream alone
        snap = gm.workspace.clone()
    st.synchronize()
    status, v = gm.pop(-1)
    assert status == gale.OK
    arr = gm.view_arrays(v)
    off = arr["tt_indices"].data_ptr() - gm.workspace.data_ptr()
    n = arr["tt_indices"].numel()
    assert torch.equal(snap[off:off + 4 * n].view(torch.int32), arr["tt_indices"])
    host = {k: (x.cpu().numpy() if hasattr(x, "cpu") else x) for k, x in arr.items()}
    got = gale.split_batch(host, m.dim + 1)
    ref = oracle.cluster_results(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, ids)
    for a, r in zip(got, ref):
        assert np.array_equal(a["tt"], r["tt"]) and np.array_equal(a["vt"][1], r["vt"][1])
    gm.release(v)
    gm.destroy()
