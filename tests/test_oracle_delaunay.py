"""Oracle pins on IRREGULAR meshes: Delaunay triangulations of random points (vertex degrees vary widely,
unlike the Kuhn grids of the BASELINE configs). Pinned to things that share nothing with oracle/:
  * TT  against Qhull's own simplex-adjacency array (scipy.spatial.Delaunay.neighbors: the simplex opposite
        each vertex, -1 on the hull), carried through the renumbering and canonicalisation;
  * VT  against the CSR transpose of the incidence matrix B, VV against the pattern of B Bt minus the
        diagonal (scipy.sparse);
  * the Euler characteristic of a ball, V - E + F - T = 1 (3-D) / V - E + T = 1 (2-D), with E and F
        derived from the oracle's VV and TT (SURVEY.md §8(c) "global")."""
import numpy as np
import pytest
import scipy.sparse as sp

import meshgen
import oracle

CASES = [(3, 1500, 11, 300), (3, 4000, 12, 700), (2, 6000, 13, 500), (2, 300, 14, 64)]


def _global(m):
    ids = list(range(m.num_clusters))
    res = oracle.cluster_results(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, ids)
    cat = lambda k: (np.concatenate([[0], np.cumsum(np.concatenate([np.diff(r[k][0]) for r in res]))]),
                     np.concatenate([r[k][1] for r in res]))
    return cat("vt"), cat("vv"), np.concatenate([r["tt"] for r in res])


@pytest.mark.parametrize("dim,npts,seed,cap", CASES)
def test_tt_equals_qhull_neighbors(dim, npts, seed, cap):
    m = meshgen.make_delaunay(dim, npts, seed=seed, capacity=cap)
    _, _, tt = _global(m)
    rank, perm = m.meta["vertex_rank"], m.meta["simplex_perm"]
    qs, qn = m.meta["qhull_simplices"][perm], m.meta["qhull_neighbors"][perm]    # canonical simplex order
    inv = np.empty(len(perm), np.int64)
    inv[perm] = np.arange(len(perm))
    j = np.argsort(rank[qs], axis=1)                   # canonical position k holds original position j[k]
    assert np.array_equal(np.take_along_axis(rank[qs], j, axis=1), m.simplices)
    nb = np.take_along_axis(qn, j, axis=1)
    want = np.where(nb >= 0, inv[np.maximum(nb, 0)], -1)
    assert np.array_equal(tt, want)


@pytest.mark.parametrize("dim,npts,seed,cap", CASES)
def test_vt_vv_sparse_and_euler(dim, npts, seed, cap):
    m = meshgen.make_delaunay(dim, npts, seed=seed, capacity=cap)
    (vto, vti), (vvo, vvi), tt = _global(m)
    T, nV, nT, D = m.simplices, m.num_vertices, m.num_simplices, m.dim + 1
    B = sp.csr_matrix((np.ones(nT * D, np.int8), (T.ravel(), np.repeat(np.arange(nT), D))), shape=(nV, nT))
    B.sort_indices()
    assert np.array_equal(vto, B.indptr) and np.array_equal(vti, B.indices)
    A = (B.astype(np.int32) @ B.astype(np.int32).T).tolil()
    A.setdiag(0)
    A = A.tocsr()
    A.eliminate_zeros()
    A.sort_indices()
    assert np.array_equal(vvo, A.indptr) and np.array_equal(vvi, A.indices)
    E, boundary = len(vvi) // 2, int((tt == -1).sum())
    if dim == 3:
        F = (4 * nT + boundary) // 2
        assert (4 * nT + boundary) % 2 == 0 and nV - E + F - nT == 1
    else:
        assert (3 * nT + boundary) == 2 * E and nV - E + nT == 1
    deg = np.diff(vto)                                                  # sanity of the test mesh itself:
    assert deg.max() >= 1.5 * deg.mean() and deg.min() < deg.mean()     # vertex degrees are far from uniform
