"""Pins of the CPU oracle against things other than itself (SURVEY.md §8(c) pin table).

Each test is chosen so that a plausible mistake in oracle/gale_oracle.cpp (dropped term, wrong
index, transposed operand, self not excluded, wrong facet <-> opposite-vertex order) fails it.
All CPU-only.
"""
import os

import numpy as np
import pytest
import scipy.sparse as sp

import meshgen
import oracle


def rows(off, idx):
    return [idx[off[i]:off[i + 1]].tolist() for i in range(len(off) - 1)]


# ---------------------------------------------------------------- golden: Fig. 1 toy
def _read_fig1(golden_dir):
    simp, exp = [], {"VV": {}, "VT": {}, "TT": {}}
    for line in open(os.path.join(golden_dir, "fig1_toy.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        head, vals = line.split(":")
        head = head.split()
        vals = [int(x) for x in vals.split()]
        if head[0] == "simplices":
            simp.append(vals)
        else:
            exp[head[1]][int(head[2])] = vals
    return np.array(simp, np.int32), exp


def test_fig1_toy_golden(golden_dir):
    T, exp = _read_fig1(golden_dir)
    R = oracle.relations_global(3, 5, T)
    vv, vt = rows(R["vv_off"], R["vv_idx"]), rows(R["vt_off"], R["vt_idx"])
    assert vv[0] == [1, 2, 3]                      # the value the paper prints
    for v, e in exp["VV"].items():
        assert vv[v] == e
    for v, e in exp["VT"].items():
        assert vt[v] == e
    for t, e in exp["TT"].items():
        assert R["tt"][t].tolist() == e


# ---------------------------------------------------------------- brute force on tiny meshes
TINY = [
    dict(dim=3, n=4),
    dict(dim=3, n=5, drop_frac=0.15),
    dict(dim=3, n=5, clustering="octree", capacity=20, permute=True),
    dict(dim=3, n=5, clustering="octree", capacity=16, warp=True, drop_frac=0.3),
    dict(dim=2, n=8, clustering="morton", block=4),
    dict(dim=2, n=9, clustering="octree", capacity=10, permute=True, drop_frac=0.2),
]


@pytest.mark.parametrize("spec", TINY)
def test_brute_force(spec):
    spec = dict(spec)
    if spec.get("clustering", "morton") == "morton":
        spec.setdefault("block", 2 if spec["n"] % 2 == 0 else 1)
        if spec["n"] & (spec["n"] - 1):
            spec.update(clustering="octree", capacity=12)
    m = meshgen.make_mesh(seed=1234, **spec)
    R = oracle.relations_global(m.dim, m.num_vertices, m.simplices)
    B = oracle.brute_force(m.dim, m.num_vertices, m.simplices)
    for k in ("vt_off", "vt_idx", "vv_off", "vv_idx", "tt"):
        assert np.array_equal(R[k], B[k]), k


# ---------------------------------------------------------------- library pins (scipy.sparse)
@pytest.mark.parametrize("dim,n", [(3, 9), (2, 20)])
def test_scipy_incidence(dim, n):
    m = meshgen.make_mesh(dim, n, clustering="octree", capacity=64, permute=True, drop_frac=0.1, seed=77)
    T, nV, nT, D = m.simplices, m.num_vertices, m.num_simplices, dim + 1
    R = oracle.relations_global(dim, nV, T)
    # B = V x T incidence matrix
    B = sp.csr_matrix((np.ones(nT * D, np.int32), (T.ravel(), np.repeat(np.arange(nT), D))), shape=(nV, nT))
    B.sort_indices()
    # VT = CSR of B (= transpose of the T x V list)
    assert np.array_equal(B.indptr, R["vt_off"]) and np.array_equal(B.indices, R["vt_idx"])
    # VV = pattern of B B^T minus the diagonal
    A = (B @ B.T).tolil()
    A.setdiag(0)
    A = A.tocsr()
    A.eliminate_zeros()
    A.sort_indices()
    assert np.array_equal(A.indptr, R["vv_off"]) and np.array_equal(A.indices, R["vv_idx"])
    # TT neighbour *sets* = pairs of simplices sharing exactly D-1 vertices
    S = (B.T @ B).tocoo()
    keep = (S.data == D - 1) & (S.row != S.col)
    N = sp.csr_matrix((np.ones(keep.sum(), np.int8), (S.row[keep], S.col[keep])), shape=(nT, nT))
    N.sort_indices()
    for t in range(nT):
        got = sorted(x for x in R["tt"][t].tolist() if x >= 0)
        assert got == N.indices[N.indptr[t]:N.indptr[t + 1]].tolist()


# ---------------------------------------------------------------- closed forms, Euler, degrees
def _closed_forms(golden_dir):
    out = []
    for line in open(os.path.join(golden_dir, "kuhn_closed_forms.txt")):
        if line.startswith("#") or not line.strip():
            continue
        d, n, V, T, E, F, b = line.split()
        out.append((int(d), int(n), int(V), int(T), int(E), None if F == "-" else int(F), int(b)))
    return out


def test_kuhn_closed_forms_and_euler(golden_dir):
    for dim, n, V, nT, E, F, bnd in _closed_forms(golden_dir):
        D = dim + 1
        m = meshgen.make_mesh(dim, n, clustering="octree", capacity=50, seed=5)
        assert (m.num_vertices, m.num_simplices) == (V, nT)
        R = oracle.relations_global(dim, V, m.simplices)
        assert R["vt_off"][-1] == D * nT                      # sum |VT| = D * #simplices
        assert R["vv_off"][-1] == 2 * E                       # sum |VV| = 2 E
        nb = int((R["tt"] < 0).sum())
        assert nb == bnd                                      # boundary facets
        if dim == 3:
            assert (D * nT + nb) // 2 == F
            assert V - E + F - nT == 1                        # Euler characteristic of a ball
        else:
            assert (D * nT + nb) // 2 == E                    # facets of a 2-D mesh are its edges
            assert V - E + nT == 1
        # no -1 inside VT / VV rows, self never in VV
        assert R["vt_idx"].min() >= 0 and R["vv_idx"].min() >= 0
        src = np.repeat(np.arange(V), np.diff(R["vv_off"]))
        assert not np.any(src == R["vv_idx"])


@pytest.mark.parametrize("dim,n,dvt,dvv", [(3, 7, 24, 14), (2, 12, 6, 6)])
def test_interior_kuhn_degrees(dim, n, dvt, dvv):
    m = meshgen.make_mesh(dim, n, clustering="octree", capacity=40, permute=True, seed=9)
    R = oracle.relations_global(dim, m.num_vertices, m.simplices)
    g2f = m.meta["grid_to_final"]
    g = np.arange(n ** dim)
    coords = np.stack([(g // n ** a) % n for a in range(dim)], 1)
    interior = np.all((coords > 0) & (coords < n - 1), axis=1)
    vs = g2f[interior]
    assert np.all(np.diff(R["vt_off"])[vs] == dvt)
    assert np.all(np.diff(R["vv_off"])[vs] == dvv)


# ---------------------------------------------------------------- structural invariants of TT
@pytest.mark.parametrize("dim,n,drop", [(3, 10, 0.0), (3, 10, 0.15), (2, 30, 0.15)])
def test_tt_symmetry_and_shared_facet(dim, n, drop):
    m = meshgen.make_mesh(dim, n, clustering="octree", capacity=100, drop_frac=drop, seed=3)
    T, D = m.simplices, dim + 1
    tt = oracle.relations_global(dim, m.num_vertices, T, mask=oracle.REL_TT)["tt"]
    for k in range(D):
        t = np.nonzero(tt[:, k] >= 0)[0]
        s = tt[t, k]
        assert np.all(s != t)
        facet = np.delete(T[t], k, axis=1)                    # T[t] minus its k-th vertex
        # every facet vertex lies in the neighbour, and the neighbour points back through the same facet
        for j in range(D - 1):
            assert np.all((T[s] == facet[:, j:j + 1]).any(axis=1))
        back = (tt[s] == t[:, None])
        assert np.all(back.sum(axis=1) == 1)
        kk = back.argmax(axis=1)
        other = np.stack([np.delete(T[si], ki) for si, ki in zip(s, kk)]) if len(s) else facet
        assert np.array_equal(other, facet)
        # |T[t] ∩ T[s]| = D-1 exactly
        inter = sum((T[t][:, a:a + 1] == T[s]).any(axis=1).astype(int) for a in range(D))
        assert np.all(inter == D - 1)


def test_vv_symmetry_and_star_union():
    m = meshgen.make_mesh(3, 8, clustering="octree", capacity=64, warp=True, drop_frac=0.1, seed=11)
    R = oracle.relations_global(3, m.num_vertices, m.simplices)
    vv, vt = rows(R["vv_off"], R["vv_idx"]), rows(R["vt_off"], R["vt_idx"])
    pairs = {(v, u) for v in range(m.num_vertices) for u in vv[v]}
    assert all((u, v) in pairs for (v, u) in pairs)
    for v in range(m.num_vertices):                          # VV(v) = union of VT(v)'s vertices minus v
        star = set(m.simplices[vt[v]].ravel().tolist()) - {v}
        assert sorted(star) == vv[v]


# ---------------------------------------------------------------- clustering independence
def test_clustering_independence():
    a = meshgen.make_mesh(3, 8, clustering="morton", block=4, seed=21, keep_fields=True)
    b = meshgen.make_mesh(3, 8, clustering="octree", capacity=30, permute=True, seed=22, keep_fields=True)
    Ra = oracle.relations_global(3, a.num_vertices, a.simplices)
    Rb = oracle.relations_global(3, b.num_vertices, b.simplices)
    ga, gb = a.meta["grid_to_final"], b.meta["grid_to_final"]
    a2b = np.empty_like(ga)
    a2b[ga] = gb                                              # vertex id in a -> vertex id in b
    # simplex id in a -> simplex id in b via the canonical row
    key = lambda T: [tuple(r) for r in T.tolist()]
    where_b = {r: i for i, r in enumerate(key(b.simplices))}
    ta2b = np.array([where_b[tuple(sorted(a2b[r].tolist()))] for r in a.simplices])
    vva, vvb = rows(Ra["vv_off"], Ra["vv_idx"]), rows(Rb["vv_off"], Rb["vv_idx"])
    vta, vtb = rows(Ra["vt_off"], Ra["vt_idx"]), rows(Rb["vt_off"], Rb["vt_idx"])
    for v in range(a.num_vertices):
        assert sorted(a2b[vva[v]].tolist()) == vvb[a2b[v]]
        assert sorted(ta2b[vta[v]].tolist()) == vtb[a2b[v]]
    for t in range(a.num_simplices):
        na = {int(ta2b[x]) for x in Ra["tt"][t] if x >= 0}
        nb = {int(x) for x in Rb["tt"][ta2b[t]] if x >= 0}
        assert na == nb


# ---------------------------------------------------------------- per-cluster slices
def test_cluster_slices_cover_global_once():
    m = meshgen.make_config(4, n=20)
    G = oracle.relations_global(3, m.num_vertices, m.simplices)
    res = oracle.cluster_results(3, m.num_vertices, m.simplices, m.cluster_offsets, range(m.num_clusters))
    vt_i = np.concatenate([r["vt"][1] for r in res])
    vv_i = np.concatenate([r["vv"][1] for r in res])
    tt = np.concatenate([r["tt"] for r in res])
    assert np.array_equal(vt_i, G["vt_idx"]) and np.array_equal(vv_i, G["vv_idx"]) and np.array_equal(tt, G["tt"])
    t_next = 0
    for r in res:                                            # internal ranges tile [0, nT) in order
        assert r["t_lo"] == t_next and r["tt"].shape[0] == r["t_hi"] - r["t_lo"]
        t_next = r["t_hi"]
        assert r["vt"][0][0] == 0 and r["vt"][0][-1] == len(r["vt"][1])
        if r["t_hi"] > r["t_lo"]:                            # internal iff lowest vertex in the cluster
            v0 = m.simplices[r["t_lo"]:r["t_hi"], 0]
            assert v0.min() >= r["v_lo"] and v0.max() < r["v_hi"]
    assert t_next == m.num_simplices


@pytest.mark.parametrize("cfg,n", [(3, 24), (4, 24), (2, 96), (1, None)])
def test_restricted_equals_global_slice(cfg, n):
    m = meshgen.make_config(cfg, n=n)
    rng = np.random.default_rng(cfg)
    sel = rng.choice(m.num_clusters, size=min(5, m.num_clusters), replace=False).tolist()
    a = oracle.cluster_results(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, sel)
    b = oracle.cluster_results(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, sel, restricted=True)
    for ra, rb in zip(a, b):
        assert (ra["t_lo"], ra["t_hi"]) == (rb["t_lo"], rb["t_hi"])
        for k in ("vt", "vv"):
            assert np.array_equal(ra[k][0], rb[k][0]) and np.array_equal(ra[k][1], rb[k][1])
        assert np.array_equal(ra["tt"], rb["tt"])


# ---------------------------------------------------------------- contract violations are refused
def test_rejects_bad_input():
    m = meshgen.make_mesh(3, 4, seed=2, block=2)
    T = m.simplices.copy()
    T[[3, 4]] = T[[4, 3]]                                     # rows out of lexicographic order
    with pytest.raises(oracle.OracleError):
        oracle.relations_global(3, m.num_vertices, T)
    T = m.simplices.copy()
    T[0, 0], T[0, 1] = T[0, 1], T[0, 0]                       # row not ascending
    with pytest.raises(oracle.OracleError):
        oracle.relations_global(3, m.num_vertices, T)
    # three triangles on one edge: non-manifold facet
    T = np.array([[0, 1, 2], [0, 1, 3], [0, 1, 4]], np.int32)
    with pytest.raises(oracle.OracleError):
        oracle.relations_global(2, 5, T)


# ---- initialization data: I_T and T_ex -------------------------------------------
def _fig4(golden_dir):
    T, S, exp = [], [], {}
    for line in open(os.path.join(golden_dir, "fig4_mesh.txt")):
        f = line.split()
        if not f or f[0].startswith("#"):
            continue
        if f[0] == "T":
            T.append([int(x) for x in f[1:]])
        elif f[0] == "S":
            S.append((int(f[1]), int(f[2])))
        else:
            exp[f[0]] = [int(x) for x in f[1:]]
    return np.array(T, np.int32), S, exp


def test_fig4_internal_external_and_edge_intervals(golden_dir):
    """The paper's own statements about its Fig. 4 example: t1 internal to S1 / external to S2, and the
    edge interval array I_E = [0, 9, 12] (9 edges with their lowest vertex in S1, 3 in S2)."""
    T, S, exp = _fig4(golden_dir)
    ranges = [oracle.internal_range(3, T, lo, hi) for lo, hi in S]
    assert [ranges[0][0], ranges[0][1], ranges[1][1]] == exp["I_T"] and ranges[1][0] == ranges[0][1]
    assert ranges[0][0] <= 1 < ranges[0][1]                          # t1 is internal to S1
    assert oracle.external_list(3, T, *S[0]).tolist() == exp["TEX_S1"]
    tex2 = oracle.external_list(3, T, *S[1]).tolist()
    assert tex2 == exp["TEX_S2"] and 1 in tex2                       # ... and external to S2
    # I_E from the VV relation: an edge is internal to the segment of its lower vertex
    g = oracle.relations_global(3, 6, T, mask=2)
    per_seg = [sum(int((g["vv_idx"][g["vv_off"][v]:g["vv_off"][v + 1]] > v).sum()) for v in range(lo, hi)) for lo, hi in S]
    assert [0, per_seg[0], per_seg[0] + per_seg[1]] == exp["I_E"]


@pytest.mark.parametrize("dim,n,seed", [(3, 7, 3), (2, 12, 4)])
def test_internal_external_brute_force(dim, n, seed):
    """I_T / T_ex against set arithmetic on small meshes with holes: the segments' internal ranges tile
    [0, nT); internal + external = every simplex touching the segment; no simplex is both."""
    m = meshgen.make_mesh(dim, n, clustering="octree", capacity=40, permute=True, drop_frac=0.2, seed=seed)
    T = m.simplices
    prev = 0
    for c in range(m.num_clusters):
        lo, hi = int(m.cluster_offsets[c]), int(m.cluster_offsets[c + 1])
        a, b = oracle.internal_range(dim, T, lo, hi)
        assert a == prev and b >= a
        prev = b
        ext = oracle.external_list(dim, T, lo, hi)
        touching = {t for t in range(len(T)) if any(lo <= v < hi for v in T[t])}
        internal = {t for t in range(len(T)) if lo <= min(T[t]) < hi}
        assert set(range(a, b)) == internal
        assert ext.tolist() == sorted(touching - internal)
    assert prev == len(T)


# ---- edges, triangles, VE, VF (Table 1) --------------------------------------------------
def test_fig4_edge_list_and_interval_array(golden_dir):
    """The paper's Fig. 4/5 example: 12 edges with I_E = [0, 9, 12]; edge (v0, v3) is e2 and
    (v3, v4) is e9 (:192). [(v0, v4) = e6 in the paper cannot hold in ANY list sorted by vertex indices that
    also has (v0, v3) = e2 — the mesh of the figure is not in the text; DESIGN.md §2 reading 18.]"""
    T, S, exp = _fig4(golden_dir)
    e = oracle.sub_simplices(3, 6, T, 2)
    assert len(e["list"]) == 12
    assert [int(e["first"][S[0][0]]), int(e["first"][S[1][0]]), int(e["first"][6])] == exp["I_E"]
    assert e["list"][2].tolist() == [0, 3] and e["list"][9].tolist() == [3, 4]
    f = oracle.sub_simplices(3, 6, T, 3)
    assert [0, 3, 4] in f["list"].tolist()                          # the triangle f5 of the FE example exists


@pytest.mark.parametrize("dim,n", [(3, 6), (2, 9)])
def test_edges_triangles_closed_forms_and_brute_force(dim, n):
    m = meshgen.make_mesh(dim, n, clustering="octree", capacity=60, permute=True, seed=21)
    T, nV = m.simplices, m.num_vertices
    cf = meshgen.kuhn_closed_forms(dim, n)
    e = oracle.sub_simplices(dim, nV, T, 2)
    f = oracle.sub_simplices(dim, nV, T, 3)
    assert len(e["list"]) == cf["E"]
    assert len(f["list"]) == (cf["F"] if dim == 3 else cf["T"])
    if dim == 2:
        assert np.array_equal(f["list"], T)                          # in 2-D the triangles are the simplices
    # brute force with python sets
    edges = sorted({(int(r[i]), int(r[j])) for r in T for i in range(dim + 1) for j in range(i + 1, dim + 1)})
    assert e["list"].tolist() == [list(x) for x in edges]
    tris = sorted({tuple(int(x) for x in np.delete(r, k)) for r in T for k in range(dim + 1)}) if dim == 3 else [tuple(r) for r in T.tolist()]
    assert f["list"].tolist() == [list(x) for x in tris]
    g = oracle.relations_global(dim, nV, T, mask=3)
    for s, name in ((e, "VE"), (f, "VF")):
        k = s["list"].shape[1]
        assert s["v_off"][-1] == k * len(s["list"])                  # sum |VE| = 2 E, sum |VF| = 3 F
        assert (np.diff(s["first"]) >= 0).all() and s["first"][-1] == len(s["list"])
        assert np.array_equal(np.searchsorted(s["list"][:, 0], np.arange(nV + 1)), s["first"])
        for v in (0, nV // 2, nV - 1):
            row = s["v_idx"][s["v_off"][v]:s["v_off"][v + 1]]
            assert (np.diff(row) > 0).all()
            assert row.tolist() == [i for i, x in enumerate(s["list"].tolist()) if v in x]
    assert np.array_equal(np.diff(e["v_off"]), np.diff(g["vv_off"]))  # |VE(v)| = |VV(v)|
    # VE(v)[i] is the edge (v, VV(v)[i]): edge ids ascend with the neighbour
    v = nV // 2
    nb = g["vv_idx"][g["vv_off"][v]:g["vv_off"][v + 1]]
    ev = e["list"][e["v_idx"][e["v_off"][v]:e["v_off"][v + 1]]]
    assert np.array_equal(np.where(ev[:, 0] == v, ev[:, 1], ev[:, 0]), nb)
    if dim == 3:
        assert np.diff(f["v_off"]).max() == 36                        # interior Kuhn vertex: 36 triangles


@pytest.mark.parametrize("n", [5, 7])
def test_ef_et_ft_counts_brute_force_and_tt_consistency(n):
    """EF / ET / FT (Table 1): closed-form sums, python-set brute force, and FT against TT —
    a triangle with two cofaces is exactly a pair of face-adjacent simplices."""
    m = meshgen.make_mesh(3, n, clustering="octree", capacity=80, permute=True, seed=31)
    T, nV, nT = m.simplices, m.num_vertices, m.num_simplices
    cf = meshgen.kuhn_closed_forms(3, n)
    E = oracle.sub_simplices(3, nV, T, 2)["list"]
    F = oracle.sub_simplices(3, nV, T, 3)["list"]
    et = oracle.coboundary(3, nV, T, "ET")
    ft = oracle.coboundary(3, nV, T, "FT")
    ef = oracle.coboundary(3, nV, T, "EF")
    assert et[0][-1] == 6 * nT and ft[0][-1] == 4 * nT and ef[0][-1] == 3 * len(F)       # incidences counted from the other side
    assert len(et[0]) - 1 == len(E) and len(ft[0]) - 1 == len(F) == len(ef[0]) - 1 + len(F) - len(E)
    nft = np.diff(ft[0])
    assert set(nft.tolist()) <= {1, 2} and int((nft == 1).sum()) == cf["boundary_facets"]
    sets = [set(r.tolist()) for r in T]
    for rows, (off, idx), cols in ((E, et, sets), (F, ft, sets), (E, ef, [set(r.tolist()) for r in F])):
        for r in (0, len(rows) // 3, len(rows) - 1):
            want = [i for i, c in enumerate(cols) if set(rows[r].tolist()) <= c]
            assert idx[off[r]:off[r + 1]].tolist() == want
    tt = oracle.relations_global(3, nV, T, mask=4)["tt"]
    pairs_tt = {(min(t, int(u)), max(t, int(u))) for t in range(nT) for u in tt[t] if u >= 0}
    pairs_ft = {(int(ft[1][ft[0][f]]), int(ft[1][ft[0][f] + 1])) for f in range(len(F)) if nft[f] == 2}
    assert pairs_tt == pairs_ft


# ---- canonical form (SURVEY.md §8(f)-1 "canonicalisation itself"; DESIGN.md §2 reading 2) ------------------
def _scramble(T, seed):
    """Rows in random order, vertices in random order inside every row (seeded)."""
    rng = np.random.default_rng(seed)
    rows = T[rng.permutation(len(T))]
    cols = np.argsort(rng.random(rows.shape), axis=1)
    return np.take_along_axis(rows, cols, axis=1)


@pytest.mark.parametrize("make", [lambda: meshgen.make_config(1), lambda: meshgen.make_mesh(2, 40, clustering="morton", block=8),
                                  lambda: meshgen.make_delaunay(3, 800, seed=9, capacity=200)],
                         ids=["kuhn3d", "grid2d", "delaunay3d"])
def test_canonical_form_pins(make):
    m = make()
    T = m.simplices
    S = _scramble(T, 17)
    got, perm = oracle.canonical_form(S)
    # (1) the generator canonicalises with its own C++ code: a scrambled copy must come back to exactly its output
    assert np.array_equal(got, T)
    # (2) plain Python: sorted tuples of sorted rows
    assert [tuple(r) for r in got] == sorted(tuple(sorted(r)) for r in S.tolist())
    # (3) the permutation leads back to the input rows, and a canonical list is a fixed point
    assert np.array_equal(np.sort(S[perm], axis=1), got) and sorted(perm.tolist()) == list(range(len(S)))
    again, p2 = oracle.canonical_form(T)
    assert np.array_equal(again, T) and np.array_equal(p2, np.arange(len(T)))
    # (4) the oracle's own C1 / C2 check (its C++ input contract) accepts it and rejects the scrambled list
    oracle.relations_global(m.dim, m.num_vertices, got, mask=1)
    with pytest.raises(oracle.OracleError):
        oracle.relations_global(m.dim, m.num_vertices, S, mask=1)


def test_canonical_form_is_stable_on_equal_rows():
    S = np.array([[5, 1, 3, 2], [0, 9, 4, 7], [2, 5, 1, 3], [3, 2, 1, 5], [7, 9, 0, 4]], dtype=np.int32)
    got, perm = oracle.canonical_form(S)
    assert got.tolist() == [[0, 4, 7, 9], [0, 4, 7, 9], [1, 2, 3, 5], [1, 2, 3, 5], [1, 2, 3, 5]]
    assert perm.tolist() == [1, 4, 0, 2, 3]   # equal rows keep their input order


# ---- boundary relations FE / TE / TF (Table 1 :53-58; look-up :186-192) ---------------------------
def test_fig4_fe_example(golden_dir):
    """FE of the triangle (v0, v3, v4) ('f5'): edges (v0,v3), (v0,v4), (v3,v4) in this order; the
    paper prints e2, e6, e9 — e2 and e9 are reproduced, e6 cannot be (DESIGN.md §2 reading 18)."""
    T, S, exp = _fig4(golden_dir)
    F = oracle.sub_simplices(3, 6, T, 3)["list"].tolist()
    fe = oracle.boundary(3, 6, T, "FE")
    row = fe[F.index([0, 3, 4])].tolist()
    assert row[0] == 2 and row[2] == 9
    E = oracle.sub_simplices(3, 6, T, 2)["list"].tolist()
    assert [E[e] for e in row] == [[0, 3], [0, 4], [3, 4]]


@pytest.mark.parametrize("make", [lambda: meshgen.make_mesh(3, 6, clustering="octree", capacity=60, permute=True, seed=21),
                                  lambda: meshgen.make_mesh(3, 7, clustering="octree", capacity=80, drop_frac=0.2, seed=4),
                                  lambda: meshgen.make_delaunay(3, 300, seed=12, capacity=80)], ids=["kuhn", "holes", "delaunay"])
def test_boundary_relations_are_transposes_of_the_coboundary_relations(make):
    m = make()
    T, nV = m.simplices, m.num_vertices
    for bnd, cob in (("FE", "EF"), ("TE", "ET"), ("TF", "FT")):
        B = oracle.boundary(3, nV, T, bnd)
        off, idx = oracle.coboundary(3, nV, T, cob)      # rows = sub-simplices, entries = containing simplices
        pairs_b = {(int(x), r) for r, row in enumerate(B.tolist()) for x in row}
        pairs_c = {(r, int(x)) for r in range(len(off) - 1) for x in idx[off[r]:off[r + 1]]}
        assert pairs_b == pairs_c, bnd
        assert all(len(set(row)) == B.shape[1] for row in B.tolist())    # distinct faces
    assert oracle.boundary(3, nV, T, "TE").shape == (len(T), 6) and oracle.boundary(3, nV, T, "TF").shape == (len(T), 4)


def test_boundary_te_2d():
    m = meshgen.make_mesh(2, 9, clustering="octree", capacity=30, seed=2)
    te = oracle.boundary(2, m.num_vertices, m.simplices, "TE")
    E = oracle.sub_simplices(2, m.num_vertices, m.simplices, 2)["list"]
    for t, row in zip(m.simplices.tolist(), te.tolist()):   # brute force: position of each pair in the sorted edge list
        assert [E[e].tolist() for e in row] == [[t[0], t[1]], [t[0], t[2]], [t[1], t[2]]]
