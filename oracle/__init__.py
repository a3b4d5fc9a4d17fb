"""oracle — CPU oracle of the GALE relation hot path. TEST INFRASTRUCTURE ONLY.

ctypes wrapper over oracle/gale_oracle.cpp (plain single-threaded C++; see its header for the
definitions, citations and pins). Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference leg may import this package. It never imports the CUDA package
(paper_2507_15230_b200) and shares no code with it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gale_oracle.cpp")
_LIB = os.path.join(_HERE, "libgale_oracle.so")
_lib = None

REL_VT, REL_VV, REL_TT = 1, 2, 4


def build(force: bool = False) -> str:
    """Compile gale_oracle.cpp -> libgale_oracle.so (g++ -O2, host only, no SIMD tricks)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp, i64, c_int, u32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_uint32
        i32p, i64p = ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int64)
        lib.go_compute_global.restype = vp
        lib.go_compute_global.argtypes = [c_int, i64, i64, i32p, u32]
        lib.go_status.restype = c_int
        lib.go_status.argtypes = [vp]
        lib.go_free.restype = None
        lib.go_free.argtypes = [vp]
        for name, rt in [("go_vt_offsets", i64p), ("go_vt_indices", i32p), ("go_vv_offsets", i64p),
                         ("go_vv_indices", i32p), ("go_tt", i32p), ("go_first_tet", i64p)]:
            getattr(lib, name).restype = rt
            getattr(lib, name).argtypes = [vp]
        lib.go_vv_nnz.restype = i64
        lib.go_vv_nnz.argtypes = [vp]
        lib.go_compute_restricted.restype = vp
        lib.go_compute_restricted.argtypes = [c_int, i64, i64, i32p, ctypes.c_int32, i32p, ctypes.c_int32, i32p, u32]
        lib.go_sub_relations.restype = vp
        lib.go_sub_relations.argtypes = [vp]
        lib.go_sub_gid.restype = i32p
        lib.go_sub_gid.argtypes = [vp]
        lib.go_sub_size.restype = i64
        lib.go_sub_size.argtypes = [vp]
        lib.go_seconds.restype = None
        lib.go_seconds.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
        lib.go_sub_extract_seconds.restype = ctypes.c_double
        lib.go_sub_extract_seconds.argtypes = [vp]
        lib.go_sub_free.restype = None
        lib.go_sub_free.argtypes = [vp]
        lib.go_slice_rows.restype = i64
        lib.go_slice_rows.argtypes = [i64p, i32p, i64, i64, i32p, i32p, i32p]
        lib.go_slice_tt.restype = None
        lib.go_slice_tt.argtypes = [i32p, c_int, i64, i64, i32p, i32p]
        lib.go_internal_range.restype = None
        lib.go_internal_range.argtypes = [c_int, i64, i32p, i64, i64, i64p]
        lib.go_external_list.restype = i64
        lib.go_external_list.argtypes = [c_int, i64, i32p, i64, i64, i32p]
        lib.go_enumerate_sub.restype = vp
        lib.go_enumerate_sub.argtypes = [c_int, c_int, i64, i64, i32p]
        lib.go_sub_count.restype = i64
        lib.go_sub_count.argtypes = [vp]
        lib.go_sub_list.restype = i32p
        lib.go_sub_list.argtypes = [vp]
        for name in ("go_sub_first", "go_sub_v_off"):
            getattr(lib, name).restype = i64p
            getattr(lib, name).argtypes = [vp]
        lib.go_sub_v_idx.restype = i32p
        lib.go_sub_v_idx.argtypes = [vp]
        lib.go_sub_release.restype = None
        lib.go_sub_release.argtypes = [vp]
        lib.go_coboundary.restype = vp
        lib.go_coboundary.argtypes = [c_int, c_int, c_int, i64, i64, i32p]
        lib.go_cob_rows.restype = i64
        lib.go_cob_rows.argtypes = [vp]
        lib.go_cob_off.restype = i64p
        lib.go_cob_off.argtypes = [vp]
        lib.go_cob_idx.restype = i32p
        lib.go_cob_idx.argtypes = [vp]
        lib.go_cob_release.restype = None
        lib.go_cob_release.argtypes = [vp]
        lib.go_brute_vt.restype = None
        lib.go_brute_vt.argtypes = [c_int, i64, i64, i32p, i64p, i32p]
        lib.go_brute_vv.restype = None
        lib.go_brute_vv.argtypes = [c_int, i64, i64, i32p, i64p, i32p]
        lib.go_brute_tt.restype = c_int
        lib.go_brute_tt.argtypes = [c_int, i64, i32p, i32p]
        _lib = lib
    return _lib


def _i32(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def _i64(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))


def _np(ptr, n, dtype):
    if n == 0:
        return np.empty(0, dtype)
    return np.ctypeslib.as_array(ptr, shape=(n,)).astype(dtype, copy=True)


class OracleError(RuntimeError):
    pass


def _canon(T):
    T = np.ascontiguousarray(T, dtype=np.int32)
    assert T.ndim == 2 and T.shape[1] in (3, 4)
    return T


def relations_global(dim: int, num_vertices: int, simplices: np.ndarray, mask: int = 7) -> dict:
    """Global VT / VV (CSR, int64 offsets) and TT ([nT, D]) straight from the definitions."""
    lib = _load()
    T = _canon(simplices)
    D, nT, nV = dim + 1, T.shape[0], int(num_vertices)
    h = lib.go_compute_global(dim, nV, nT, _i32(T), mask)
    try:
        st = lib.go_status(h)
        if st != 0:
            raise OracleError(f"oracle input contract violated: status {st}")
        out = dict(first_tet=_np(lib.go_first_tet(h), nV + 1, np.int64))
        if mask & REL_VT:
            out["vt_off"] = _np(lib.go_vt_offsets(h), nV + 1, np.int64)
            out["vt_idx"] = _np(lib.go_vt_indices(h), nT * D, np.int32)
        if mask & REL_VV:
            out["vv_off"] = _np(lib.go_vv_offsets(h), nV + 1, np.int64)
            out["vv_idx"] = _np(lib.go_vv_indices(h), int(lib.go_vv_nnz(h)), np.int32)
        if mask & REL_TT:
            out["tt"] = _np(lib.go_tt(h), nT * D, np.int32).reshape(nT, D)
        return out
    finally:
        lib.go_free(h)


def _slice_clusters(lib, h, D, offsets, clusters, mask, first_tet, gid, gid_first_tet):
    """Per-cluster results: VT/VV rows of the cluster's vertices, TT rows of its
    internal simplices; ids global; CSR offsets int32 starting at 0."""
    res = []
    gp = _i32(gid) if gid is not None else None
    for c in clusters:
        lo, hi = int(offsets[c]), int(offsets[c + 1])
        r = dict(cluster=int(c), v_lo=lo, v_hi=hi)
        for key, bit, fo, fi in (("vt", REL_VT, lib.go_vt_offsets, lib.go_vt_indices),
                                 ("vv", REL_VV, lib.go_vv_offsets, lib.go_vv_indices)):
            if not mask & bit:
                continue
            off = np.empty(hi - lo + 1, np.int32)
            nnz = int(lib.go_slice_rows(fo(h), fi(h), lo, hi, None, _i32(off), None))
            idx = np.empty(nnz, np.int32)
            lib.go_slice_rows(fo(h), fi(h), lo, hi, gp if key == "vt" else None, _i32(off), _i32(idx))
            r[key] = (off, idx)
        # internal simplices: contiguous range by C2 (I_T)
        t_lo, t_hi = int(first_tet[lo]), int(first_tet[hi])          # ids in the handle's mesh
        r["t_lo"] = int(gid_first_tet[lo])                           # global id of the first internal simplex
        r["t_hi"] = r["t_lo"] + (t_hi - t_lo)
        if mask & REL_TT:
            tt = np.empty((t_hi - t_lo, D), np.int32)
            lib.go_slice_tt(lib.go_tt(h), D, t_lo, t_hi, gp, _i32(tt))
            r["tt"] = tt
        res.append(r)
    return res


last_timing: dict = {}   # wall seconds of the last cluster_results call: extract (sub-mesh scans), vt, vv, tt, sub_simplices


def _timing(lib, h, extract=0.0, sub=0):
    t = (ctypes.c_double * 3)()
    lib.go_seconds(h, t)
    last_timing.clear()
    last_timing.update(extract=float(extract), vt=t[0], vv=t[1], tt=t[2], sub_simplices=int(sub))


def cluster_results(dim: int, num_vertices: int, simplices: np.ndarray, cluster_offsets: np.ndarray,
                    clusters, mask: int = 7, restricted: bool = False) -> list:
    """Oracle output for each cluster id in `clusters`, in that order.

    restricted=False: global pass then slice. restricted=True: the definitions on the sub-mesh of
    simplices meeting the selection's vertex closure (exact; see gale_oracle.cpp) — for meshes too
    large for a global pass.
    """
    lib = _load()
    T = _canon(simplices)
    D, nT, nV = dim + 1, T.shape[0], int(num_vertices)
    offsets = np.ascontiguousarray(cluster_offsets, dtype=np.int32)
    clusters = [int(c) for c in clusters]
    # first_tet of the *global* mesh (needed to name the internal range in global ids)
    gfirst = np.searchsorted(T[:, 0], np.arange(nV + 1), side="left").astype(np.int64) if nT else np.zeros(nV + 1, np.int64)
    if not restricted:
        h = lib.go_compute_global(dim, nV, nT, _i32(T), mask)
        try:
            if lib.go_status(h) != 0:
                raise OracleError(f"oracle input contract violated: status {lib.go_status(h)}")
            first = _np(lib.go_first_tet(h), nV + 1, np.int64)
            _timing(lib, h, 0.0, nT)
            return _slice_clusters(lib, h, D, offsets, clusters, mask, first, None, gfirst)
        finally:
            lib.go_free(h)
    sel = np.asarray(sorted(set(clusters)), np.int32)
    s = lib.go_compute_restricted(dim, nV, nT, _i32(T), len(offsets) - 1, _i32(offsets), len(sel), _i32(sel), mask)
    try:
        h = lib.go_sub_relations(s)
        if lib.go_status(h) != 0:
            raise OracleError(f"oracle input contract violated: status {lib.go_status(h)}")
        gid = _np(lib.go_sub_gid(s), int(lib.go_sub_size(s)), np.int32)
        first = _np(lib.go_first_tet(h), nV + 1, np.int64)
        _timing(lib, h, lib.go_sub_extract_seconds(s), len(gid))
        return _slice_clusters(lib, h, D, offsets, clusters, mask, first, gid, gfirst)
    finally:
        lib.go_sub_free(s)


def internal_range(dim: int, simplices: np.ndarray, lo: int, hi: int) -> tuple:
    """I_T of the segment [lo, hi): (first, last+1) internal simplex."""
    T = _canon(simplices)
    out = np.zeros(2, np.int64)
    _load().go_internal_range(dim, T.shape[0], _i32(T), int(lo), int(hi), _i64(out))
    return int(out[0]), int(out[1])


def external_list(dim: int, simplices: np.ndarray, lo: int, hi: int) -> np.ndarray:
    """T_ex of the segment [lo, hi): ascending ids of its external simplices."""
    lib = _load()
    T = _canon(simplices)
    n = int(lib.go_external_list(dim, T.shape[0], _i32(T), int(lo), int(hi), None))
    out = np.empty(n, np.int32)
    if n:
        lib.go_external_list(dim, T.shape[0], _i32(T), int(lo), int(hi), _i32(out))
    return out


def sub_simplices(dim: int, num_vertices: int, simplices: np.ndarray, k: int) -> dict:
    """Edges (k = 2) or triangles (k = 3) of the mesh: the sorted list [n, k] (id = row), the
    interval array `first` per vertex (I_E / I_F), and the coboundary relation VE / VF as CSR over all vertices."""
    lib = _load()
    T = _canon(simplices)
    nV = int(num_vertices)
    h = lib.go_enumerate_sub(dim, k, nV, T.shape[0], _i32(T))
    try:
        n = int(lib.go_sub_count(h))
        return dict(list=_np(lib.go_sub_list(h), n * k, np.int32).reshape(n, k),
                    first=_np(lib.go_sub_first(h), nV + 1, np.int64),
                    v_off=_np(lib.go_sub_v_off(h), nV + 1, np.int64),
                    v_idx=_np(lib.go_sub_v_idx(h), n * k, np.int32))
    finally:
        lib.go_sub_release(h)


def coboundary(dim: int, num_vertices: int, simplices: np.ndarray, name: str) -> tuple:
    """EF, ET or FT (Table 1) over the whole mesh as CSR (int64 offsets, int32 indices): rows = ids of
    the sorted edge (E..) / triangle (F..) list, entries = ascending ids of the triangles (.F) / simplices (.T)
    that contain them."""
    lib = _load()
    T = _canon(simplices)
    frm, to = {"EF": (2, 3), "ET": (2, dim + 1), "FT": (3, dim + 1)}[name]
    h = lib.go_coboundary(dim, frm, to, int(num_vertices), T.shape[0], _i32(T))
    try:
        n = int(lib.go_cob_rows(h))
        off = _np(lib.go_cob_off(h), n + 1, np.int64)
        return off, _np(lib.go_cob_idx(h), int(off[-1]), np.int32)
    finally:
        lib.go_cob_release(h)


def boundary(dim: int, num_vertices: int, simplices: np.ndarray, name: str) -> np.ndarray:
    """Boundary relations FE, TE, TF (Table 1 :53-58; the look-up of :186-192) over the whole mesh as a
    fixed-width array: row i = ids (positions in the sorted lists E / F) of the edges / triangles on
    the boundary of triangle i of F (FE) or of simplex i of T (TE, TF), in the lexicographic order of their vertex
    combinations — the order of the paper's example, FE(f5) = [(v0,v3), (v0,v4), (v3,v4)] (:192). Plain definition:
    every combination is looked up in a dictionary of the whole list (no interval array involved).
    Pins (tests/test_oracle_pins.py): FE / TE / TF are the transposes of the coboundary relations EF / ET / FT (a
    different routine of the oracle, itself pinned), the paper's e2 and e9 for the triangle (v0, v3, v4) of the
    Fig. 4 fixture, row-wise vertex sets."""
    import itertools

    T = _canon(simplices)
    frm, to = {"FE": (3, 2), "TE": (dim + 1, 2), "TF": (dim + 1, 3)}[name]
    rows = T if frm == dim + 1 and name != "FE" else sub_simplices(dim, num_vertices, T, 3)["list"]
    ids = {tuple(r): i for i, r in enumerate(sub_simplices(dim, num_vertices, T, to)["list"].tolist())}
    combos = list(itertools.combinations(range(rows.shape[1]), to))   # lexicographic
    out = np.empty((rows.shape[0], len(combos)), dtype=np.int32)
    for i, r in enumerate(rows.tolist()):
        for j, c in enumerate(combos):
            out[i, j] = ids[tuple(r[k] for k in c)]
    return out


def canonical_form(simplices: np.ndarray) -> tuple:
    """The canonical form the path expects (DESIGN.md §2 reading 2; the simplices internal to a
    segment — lowest vertex in the segment — must be one contiguous range, which the interval array I_T records):
    every row ascending, rows in ascending lexicographic order, equal rows in input order. Plain definition:
    sort each row, then a stable lexicographic sort of the rows (numpy's lexsort is stable). Returns
    (canonical rows, perm) with canonical row i = sorted(input row perm[i]).
    Pins (tests/test_oracle_pins.py): the generator's own canonicalisation (independent C++), a pure-Python
    sorted() of tuples, the oracle's C1 / C2 check, stability on duplicated rows."""
    rows = np.sort(np.ascontiguousarray(simplices, dtype=np.int32), axis=1)
    D = rows.shape[1]
    order = np.lexsort(tuple(rows[:, k] for k in range(D - 1, -1, -1)))  # last key = primary = column 0
    return np.ascontiguousarray(rows[order]), order.astype(np.int64)


def brute_force(dim: int, num_vertices: int, simplices: np.ndarray) -> dict:
    """Brute-force enumeration of VT, VV, TT for tiny meshes (membership scans only)."""
    lib = _load()
    T = _canon(simplices)
    D, nT, nV = dim + 1, T.shape[0], int(num_vertices)
    vt_off = np.empty(nV + 1, np.int64)
    vt_idx = np.empty(nT * D, np.int32)
    lib.go_brute_vt(dim, nV, nT, _i32(T), _i64(vt_off), _i32(vt_idx))
    vv_off = np.empty(nV + 1, np.int64)
    vv_idx = np.empty(nT * D * (D - 1), np.int32)
    lib.go_brute_vv(dim, nV, nT, _i32(T), _i64(vv_off), _i32(vv_idx))
    tt = np.empty((nT, D), np.int32)
    st = lib.go_brute_tt(dim, nT, _i32(T), _i32(tt))
    if st != 0:
        raise OracleError(f"non-manifold facet (status {st})")
    return dict(vt_off=vt_off, vt_idx=vt_idx[:vt_off[-1]].copy(), vv_off=vv_off,
                vv_idx=vv_idx[:vv_off[-1]].copy(), tt=tt)


def neighbour_sum(num_vertices: int, vv_off: np.ndarray, vv_idx: np.ndarray, scalar: np.ndarray) -> np.ndarray:
    """Fig. 1(c) of the paper: for each vertex, the sum of the scalar values of its adjacent
    vertices, from the oracle's own global VV. Plain loop, float64."""
    out = np.zeros(num_vertices, np.float64)
    for v in range(num_vertices):
        for u in vv_idx[vv_off[v]:vv_off[v + 1]]:
            out[v] += float(scalar[u])
    return out


CP_REGULAR, CP_MINIMUM, CP_SADDLE, CP_MAXIMUM = "regular", "minimum", "saddle", "maximum"


def critical_points(dim: int, num_vertices: int, simplices: np.ndarray, scalar: np.ndarray) -> list:
    """PL critical points of a scalar field on the vertices (the paper's CriticalPoints consumer: it
    needs VV and VT), written out as the definition: order the vertices by (scalar, id) (ties broken by id); the
    link of v is spanned by its VV neighbours, two of them adjacent when they share a simplex of VT(v); the lower
    (upper) link is the part on neighbours below (above) v. v is a minimum when its lower link is empty, a maximum
    when its upper link is empty, regular when both have exactly one connected component, a saddle otherwise.
    Components by flood fill over python sets, relations from the oracle's own global VV / VT. Slow on purpose.
    Pinned in tests/test_consumer.py: a hand-derived example on Fig. 1's two tetrahedra and the closed form for a
    linear function on a convex grid (one minimum, one maximum, no saddle).
    Returns a list of CP_* strings, one per vertex."""
    g = relations_global(dim, num_vertices, simplices, mask=3)
    T = np.asarray(simplices)
    f = [float(x) for x in np.asarray(scalar)]
    out = []
    for v in range(num_vertices):
        nb = [int(u) for u in g["vv_idx"][g["vv_off"][v]:g["vv_off"][v + 1]]]
        lower = {u for u in nb if (f[u], u) < (f[v], v)}
        adj = {u: set() for u in nb}
        for t in g["vt_idx"][g["vt_off"][v]:g["vt_off"][v + 1]]:
            others = [int(u) for u in T[int(t)] if int(u) != v]
            for a in others:
                for b in others:
                    if a != b and ((a in lower) == (b in lower)):
                        adj[a].add(b)
        comps = {True: 0, False: 0}
        seen = set()
        for u in nb:
            if u in seen:
                continue
            comps[u in lower] += 1
            seen.add(u)
            stack = [u]
            while stack:
                x = stack.pop()
                for y in adj[x]:
                    if y not in seen:
                        seen.add(y)
                        stack.append(y)
        lo, up = comps[True], comps[False]
        out.append(CP_MINIMUM if lo == 0 else CP_MAXIMUM if up == 0 else CP_REGULAR if (lo, up) == (1, 1) else CP_SADDLE)
    return out
