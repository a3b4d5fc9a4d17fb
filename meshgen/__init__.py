"""meshgen — seeded synthetic inputs for the GALE hot path (configs of BASELINE.json).

Input generators only: Kuhn grids, jitter/warp, permutation, Morton / PR-octree clustering,
renumbering, canonicalisation (SURVEY.md §8(c) C1-C3, §8(d) recipe). No VT/VV/TT arithmetic lives
here; both the CPU oracle tests and the CUDA path take their inputs from this module and from
nowhere else. The heavy loops are in meshgen.cpp (plain host C++, built on first use).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "meshgen.cpp")
_LIB = os.path.join(_HERE, "libmeshgen.so")
_lib = None

SEED_BASE = 0x6A1E0000
SUB_JITTER, SUB_SCALAR, SUB_PERM, SUB_HOLES = 0x100, 0x200, 0x300, 0x400


def build(force: bool = False) -> str:
    """Compile meshgen.cpp -> libmeshgen.so (g++, host only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i32p, f32p = ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_float)
        c_int, i64, u64 = ctypes.c_int, ctypes.c_int64, ctypes.c_uint64
        lib.mg_grid_num_vertices.restype = i64
        lib.mg_grid_num_vertices.argtypes = [c_int, c_int]
        lib.mg_grid_num_simplices.restype = i64
        lib.mg_grid_num_simplices.argtypes = [c_int, c_int]
        lib.mg_kuhn_grid.restype = None
        lib.mg_kuhn_grid.argtypes = [c_int, c_int, i32p]
        lib.mg_coords.restype = None
        lib.mg_coords.argtypes = [c_int, c_int, u64, c_int, f32p]
        lib.mg_scalar.restype = None
        lib.mg_scalar.argtypes = [i64, u64, f32p]
        lib.mg_permutation.restype = None
        lib.mg_permutation.argtypes = [i64, u64, i32p]
        lib.mg_morton_clusters.restype = ctypes.c_int32
        lib.mg_morton_clusters.argtypes = [c_int, c_int, c_int, i32p, i32p]
        lib.mg_octree_clusters.restype = ctypes.c_int32
        lib.mg_octree_clusters.argtypes = [c_int, i64, f32p, ctypes.c_int32, i32p, i32p]
        lib.mg_drop_simplices.restype = i64
        lib.mg_drop_simplices.argtypes = [c_int, i64, i32p, u64, ctypes.c_double]
        lib.mg_renumber_canonicalise.restype = None
        lib.mg_renumber_canonicalise.argtypes = [c_int, i64, i64, i32p, i32p, i32p]
        _lib = lib
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


@dataclass
class Mesh:
    """A canonical clustered mesh: the inputs of gale_mesh_create and of the oracle."""
    dim: int
    num_vertices: int
    simplices: np.ndarray            # int32 [nT, dim+1], rows ascending, rows lexicographically sorted
    cluster_offsets: np.ndarray      # int32 [nC+1], I_V: cluster c owns [o[c], o[c+1])
    coords: np.ndarray | None = None  # float32 [nV, dim], renumbered order (unused by the hot path)
    scalar: np.ndarray | None = None  # float32 [nV] (unused by the hot path)
    meta: dict = field(default_factory=dict)

    @property
    def num_simplices(self) -> int:
        return int(self.simplices.shape[0])

    @property
    def num_clusters(self) -> int:
        return int(self.cluster_offsets.shape[0] - 1)


def kuhn_closed_forms(dim: int, n: int) -> dict:
    """Closed-form simplex counts of an n^dim Kuhn grid (SURVEY.md §8(c) pins), m = n-1."""
    m = n - 1
    if dim == 3:
        return dict(V=n ** 3, T=6 * m ** 3, E=3 * n * n * m + 3 * n * m * m + m ** 3,
                    F=12 * m ** 3 + 6 * m * m, boundary_facets=12 * m * m)
    return dict(V=n * n, T=2 * m * m, E=2 * n * m + m * m, boundary_facets=4 * m)


def make_mesh(dim: int, n: int, *, clustering: str = "morton", block: int = 8, capacity: int = 4096,
              permute: bool = False, warp: bool = False, drop_frac: float = 0.0, seed: int = SEED_BASE,
              keep_fields: bool = True) -> Mesh:
    """Kuhn grid n^dim -> [permutation] -> clustering -> renumber -> canonical mesh."""
    lib = _load()
    D = dim + 1
    nV = int(lib.mg_grid_num_vertices(dim, n))
    nT = int(lib.mg_grid_num_simplices(dim, n))
    T = np.empty((nT, D), np.int32)
    lib.mg_kuhn_grid(dim, n, _p(T, ctypes.c_int32))
    coords = np.empty((nV, dim), np.float32)
    lib.mg_coords(dim, n, seed + SUB_JITTER, int(warp), _p(coords, ctypes.c_float))
    scalar = np.empty(nV, np.float32)
    lib.mg_scalar(nV, seed + SUB_SCALAR, _p(scalar, ctypes.c_float))
    if drop_frac > 0.0:
        nT = int(lib.mg_drop_simplices(dim, nT, _p(T, ctypes.c_int32), seed + SUB_HOLES, float(drop_frac)))
        T = np.ascontiguousarray(T[:nT])

    # new_id[grid vertex] accumulates the renumbering
    new_id = np.arange(nV, dtype=np.int32)
    if permute:
        perm = np.empty(nV, np.int32)
        lib.mg_permutation(nV, seed + SUB_PERM, _p(perm, ctypes.c_int32))
        new_id = perm  # grid vertex g is now called perm[g]
        inv = np.empty(nV, np.int32)
        inv[perm] = np.arange(nV, dtype=np.int32)
        coords = np.ascontiguousarray(coords[inv])
        scalar = np.ascontiguousarray(scalar[inv])

    order = np.empty(nV, np.int32)
    offsets = np.empty(nV + 1, np.int32)
    if clustering == "morton":
        if permute:
            raise ValueError("morton clustering works on grid ids; use octree with permute")
        nC = int(lib.mg_morton_clusters(dim, n, block, _p(order, ctypes.c_int32), _p(offsets, ctypes.c_int32)))
    elif clustering == "octree":
        nC = int(lib.mg_octree_clusters(dim, nV, _p(coords, ctypes.c_float), capacity,
                                        _p(order, ctypes.c_int32), _p(offsets, ctypes.c_int32)))
    else:
        raise ValueError(clustering)
    offsets = np.ascontiguousarray(offsets[:nC + 1])
    rank = np.empty(nV, np.int32)           # current id -> final id
    rank[order] = np.arange(nV, dtype=np.int32)
    new_id = rank[new_id]                   # grid id -> final id
    coords = np.ascontiguousarray(coords[order]) if keep_fields else None
    scalar = np.ascontiguousarray(scalar[order]) if keep_fields else None

    scratch = np.empty((nT, D), np.int32)
    lib.mg_renumber_canonicalise(dim, nV, nT, _p(T, ctypes.c_int32), _p(new_id, ctypes.c_int32),
                                 _p(scratch, ctypes.c_int32))
    del scratch
    meta = dict(n=n, clustering=clustering, block=block, capacity=capacity, permute=permute, warp=warp,
                drop_frac=drop_frac, seed=seed, grid_to_final=new_id if keep_fields else None)
    if drop_frac == 0.0:
        meta["closed_form"] = kuhn_closed_forms(dim, n)
    return Mesh(dim, nV, T, offsets, coords, scalar, meta)


# BASELINE.json configs 1..5 (index 0..4). `n` may be overridden to get a small mesh of the same family.
_CONFIGS = [
    dict(name="cfg1_kuhn16_morton8", dim=3, n=16, clustering="morton", block=8),
    dict(name="cfg2_tri4096_morton64", dim=2, n=4096, clustering="morton", block=64),
    dict(name="cfg3_kuhn128_perm_octree4096", dim=3, n=128, clustering="octree", capacity=4096, permute=True),
    dict(name="cfg4_kuhn192_warp_octree2048", dim=3, n=192, clustering="octree", capacity=2048, warp=True),
    dict(name="cfg5_kuhn256_octree8192", dim=3, n=256, clustering="octree", capacity=8192),
]


def config_spec(i: int) -> dict:
    return dict(_CONFIGS[i - 1])


def make_config(i: int, n: int | None = None, keep_fields: bool = False, **override) -> Mesh:
    """Config i in 1..5 of BASELINE.json; seed = 0x6A1E0000 + i."""
    spec = config_spec(i)
    name = spec.pop("name")
    if n is not None:
        spec["n"] = n
    spec.update(override)
    mesh = make_mesh(seed=SEED_BASE + i, keep_fields=keep_fields, **spec)
    mesh.meta["name"] = name if n is None else f"{name}@n={n}"
    mesh.meta["config"] = i
    return mesh


def from_simplices(dim: int, coords, simplices, *, capacity: int = 512, name: str = "user") -> Mesh:
    """Arbitrary simplicial mesh (vertex coordinates + simplices in any numbering) -> PR-octree clustering
    of the vertices -> renumbering so that clusters are contiguous id ranges -> canonical form (each simplex
    ascending, simplices in lexicographic order; DESIGN.md §2 reading 2). Input plumbing only.
    meta["vertex_rank"][old vertex] = new id; meta["simplex_perm"][new simplex] = old simplex index."""
    lib = _load()
    D = dim + 1
    coords = np.ascontiguousarray(coords, dtype=np.float32)
    simplices = np.ascontiguousarray(simplices, dtype=np.int32)
    nV = int(coords.shape[0])
    assert coords.shape == (nV, dim) and simplices.ndim == 2 and simplices.shape[1] == D
    order = np.empty(nV, np.int32)
    offsets = np.empty(nV + 1, np.int32)
    nC = int(lib.mg_octree_clusters(dim, nV, _p(coords, ctypes.c_float), capacity,
                                    _p(order, ctypes.c_int32), _p(offsets, ctypes.c_int32)))
    offsets = np.ascontiguousarray(offsets[:nC + 1])
    rank = np.empty(nV, np.int32)
    rank[order] = np.arange(nV, dtype=np.int32)
    T = np.sort(rank[simplices], axis=1)
    perm = np.lexsort(T.T[::-1]).astype(np.int64)          # rows in lexicographic order
    T = np.ascontiguousarray(T[perm], dtype=np.int32)
    meta = dict(name=name, clustering="octree", capacity=capacity, vertex_rank=rank, simplex_perm=perm)
    return Mesh(dim, nV, T, offsets, np.ascontiguousarray(coords[order]), None, meta)


def make_delaunay(dim: int, npoints: int, *, seed: int = 1, capacity: int = 512) -> Mesh:
    """Delaunay triangulation (scipy / Qhull) of seeded uniform random points in the unit cube: an
    irregular test mesh (vertex degrees vary widely, unlike a Kuhn grid) with the topology of a ball.
    meta["qhull_neighbors"] is Qhull's own simplex-adjacency array in the ORIGINAL numbering
    (neighbors[i][k] = simplex opposite vertex k of simplex i, -1 on the hull), kept so that tests can
    pin TT against an implementation that shares nothing with this repository."""
    from scipy.spatial import Delaunay

    pts = np.random.default_rng(seed).random((npoints, dim))
    tri = Delaunay(pts)
    m = from_simplices(dim, pts.astype(np.float32), tri.simplices, capacity=capacity,
                       name=f"delaunay{dim}d_{npoints}_seed{seed}")
    m.meta["qhull_simplices"] = np.asarray(tri.simplices, dtype=np.int64)
    m.meta["qhull_neighbors"] = np.asarray(tri.neighbors, dtype=np.int64)
    return m


def toy_two_tets() -> Mesh:
    """PAPER.md:60-64 (Fig. 1): two tetrahedra sharing a triangle, one cluster."""
    T = np.array([[0, 1, 2, 3], [1, 2, 3, 4]], np.int32)
    return Mesh(3, 5, T, np.array([0, 5], np.int32), meta=dict(name="fig1_toy"))
