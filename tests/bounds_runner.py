"""Run by tests/test_gpu_bounds.py in a subprocess with GALE_LIBRARY = the bounds-checked build:
a spread of meshes, tile sizes, relation masks and both local-id widths through the C ABI; prints one
line per case. Any capacity or staging-index violation surfaces as a GaleError (the device error word is
read at gale_queue_pop), which ends the process with a traceback."""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import meshgen  # noqa: E402
import oracle  # noqa: E402
import paper_2507_15230_b200 as gale  # noqa: E402

assert os.environ.get("GALE_LIBRARY", "").endswith("libgale_checked.so")

CASES = [
    ("cfg1", lambda: meshgen.make_config(1), 8, 0, 7),
    ("cfg1 VT only", lambda: meshgen.make_config(1), 8, 0, 1),
    ("cfg1 TT only", lambda: meshgen.make_config(1), 3, 0, 4),
    ("cfg2@256", lambda: meshgen.make_config(2, n=256), 5, 0, 7),
    ("cfg3@40", lambda: meshgen.make_config(3, n=40), 7, 0, 7),
    ("cfg4@40", lambda: meshgen.make_config(4, n=40), 64, 0, 7),
    ("cfg5@48", lambda: meshgen.make_config(5, n=48), 64, 0, 7),
    ("holes3d tv=7", lambda: meshgen.make_mesh(3, 14, clustering="octree", capacity=300, permute=True, drop_frac=0.1, seed=13), 9, 7, 7),
    ("holes3d tv=1", lambda: meshgen.make_mesh(3, 14, clustering="octree", capacity=300, permute=True, drop_frac=0.1, seed=13), 9, 1, 7),
    ("holes3d tv=256 (16-bit ids)", lambda: meshgen.make_mesh(3, 20, clustering="octree", capacity=2000, permute=True, drop_frac=0.05, seed=21), 4, 256, 7),
    ("tri2d tv=256 (16-bit ids)", lambda: meshgen.make_mesh(2, 120, clustering="octree", capacity=3000, seed=22), 3, 256, 7),
    ("delaunay3d", lambda: meshgen.make_delaunay(3, 4000, seed=41, capacity=500), 6, 0, 7),
    ("delaunay3d tv=5", lambda: meshgen.make_delaunay(3, 1500, seed=42, capacity=300), 6, 5, 7),
    ("delaunay2d", lambda: meshgen.make_delaunay(2, 8000, seed=43, capacity=900), 6, 0, 7),
    ("holes2d", lambda: meshgen.make_mesh(2, 150, clustering="octree", capacity=900, warp=True, drop_frac=0.2, seed=6), 16, 0, 7),
]

RUNS = [(c, k) for c in CASES for k in ("dense", "walk")]
for (name, make, batch, tv, mask), kernel in RUNS:
    m = make()
    name = f"{name} [{kernel}]"
    try:
        gm = gale.GaleMesh(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, max_batch_clusters=batch, tile_vertices=tv,
                           flags=gale.VALIDATE | (gale.KERNEL_WALK if kernel == "walk" else gale.KERNEL_DENSE))
    except gale.GaleError as e:
        if kernel == "walk" and e.status == gale.ERR_UNSUPPORTED:
            print(f"skip {name}: the walk kernel does not admit this mesh")
            continue
        raise
    ids = list(range(m.num_clusters))
    got = []
    for b in range(0, len(ids), batch):
        got += gale.split_batch(gm.run_batch(ids[b:b + batch], mask), m.dim + 1)
    if os.environ.get("GALE_CHECK_SELFTEST"):
        print("UNEXPECTED: the understated capacity was not detected", name)
        sys.exit(3)
    ref = oracle.cluster_results(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, ids, mask=mask)
    for g, r in zip(got, ref):
        for k in ("vt", "vv"):
            if k in r:
                assert np.array_equal(g[k][0], r[k][0]) and np.array_equal(g[k][1], r[k][1]), (name, k, r["cluster"])
        if "tt" in r:
            assert np.array_equal(g["tt"], r["tt"]), (name, "tt", r["cluster"])
    print(f"ok {name}: tiles {gm.info.num_tiles}, tile {gm.info.tile_vertices}, {gm.info.local_id_bytes}-byte ids")
    gm.destroy()
# VE / VF / EF / ET / FT (k_star and the list builders) through the checked build, against the oracle
SUB_CASES = [
    ("cfg1 sub", lambda: meshgen.make_config(1), 3),
    ("holes3d sub", lambda: meshgen.make_mesh(3, 16, clustering="octree", capacity=400, permute=True, drop_frac=0.15, seed=15), 5),
    ("delaunay3d sub", lambda: meshgen.make_delaunay(3, 3000, seed=44, capacity=400), 4),
]
if not os.environ.get("GALE_CHECK_SELFTEST"):
    for name, make, batch in SUB_CASES:
        m = make()
        T, nV = m.simplices, m.num_vertices
        gm = gale.GaleMesh(3, nV, T, m.cluster_offsets, max_batch_clusters=batch, device_ring=2,
                           flags=gale.VALIDATE | gale.WITH_EDGES | gale.WITH_FACETS | gale.WITH_COBOUNDARY)
        E, F = oracle.sub_simplices(3, nV, T, 2), oracle.sub_simplices(3, nV, T, 3)
        ref = {k: oracle.coboundary(3, nV, T, k.upper()) for k in ("ef", "et", "ft")}
        first = {"ef": E["first"], "et": E["first"], "ft": F["first"]}
        ids = list(range(m.num_clusters))
        mask = gale.REL_ALL | gale.REL_VE | gale.REL_VF | gale.REL_EF | gale.REL_ET | gale.REL_FT
        for b in range(0, len(ids), batch):
            for g in gale.split_batch(gm.run_batch(ids[b:b + batch], mask), 4):
                lo, hi = int(m.cluster_offsets[g["cluster"]]), int(m.cluster_offsets[g["cluster"] + 1])
                for k in ("ef", "et", "ft"):
                    off = ref[k][0][int(first[k][lo]):int(first[k][hi]) + 1]
                    assert np.array_equal(g[k][0], (off - off[0]).astype(np.int32)), (name, k, g["cluster"])
                    assert np.array_equal(g[k][1], ref[k][1][off[0]:off[-1]]), (name, k, g["cluster"])
                off = F["v_off"][lo:hi + 1]
                assert np.array_equal(g["vf"][1], F["v_idx"][off[0]:off[-1]]), (name, "vf", g["cluster"])
        print(f"ok {name}: E {gm.info.num_edges}, F {gm.info.num_triangles}")
        gm.destroy()
print("ALL CHECKED CASES PASSED")
