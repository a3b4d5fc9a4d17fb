"""Canonical form on the device (SURVEY.md §8(f)-1 "canonicalisation itself"; include/gale.h gale_canonicalize):
rows and permutation bit-exact against the oracle's plain definition (oracle.canonical_form: row sort + stable
lexicographic sort) on scrambled meshes, random rows with ids up to 2^31 - 2, duplicated rows (stability),
sizes around the 2,048-row segments of the radix passes, the empty list; degenerate rows are refused; a
scrambled config 5 (99.5 M tetrahedra) comes back to the generator's array."""
import numpy as np
import pytest

import meshgen
import oracle

pytestmark = pytest.mark.gpu


def _scramble(T, seed):
    rng = np.random.default_rng(seed)
    rows = T[rng.permutation(len(T))]
    cols = np.argsort(rng.random(rows.shape), axis=1)
    return np.ascontiguousarray(np.take_along_axis(rows, cols, axis=1))


def _check(dim, nV, S):
    import paper_2507_15230_b200 as gale

    out, perm = gale.canonicalize(dim, nV, S)
    ref, rperm = oracle.canonical_form(S)
    assert np.array_equal(out.cpu().numpy(), ref)
    assert np.array_equal(perm.cpu().numpy().astype(np.int64), rperm)
    out2, none = gale.canonicalize(dim, nV, S, want_perm=False)
    assert none is None and np.array_equal(out2.cpu().numpy(), ref)


MESHES = [
    ("cfg1", lambda: meshgen.make_config(1)),
    ("grid2d", lambda: meshgen.make_mesh(2, 70, clustering="morton", block=8)),
    ("holes3d", lambda: meshgen.make_mesh(3, 14, clustering="octree", capacity=300, permute=True, drop_frac=0.15, seed=5)),
    ("delaunay3d", lambda: meshgen.make_delaunay(3, 3000, seed=21, capacity=400)),
    ("delaunay2d", lambda: meshgen.make_delaunay(2, 5000, seed=22, capacity=500)),
]


@pytest.mark.parametrize("name,make", MESHES, ids=[c[0] for c in MESHES])
def test_scrambled_mesh_returns_to_canonical_form(name, make):
    m = make()
    S = _scramble(m.simplices, 3)
    _check(m.dim, m.num_vertices, S)
    import paper_2507_15230_b200 as gale

    out, _ = gale.canonicalize(m.dim, m.num_vertices, S)
    assert np.array_equal(out.cpu().numpy(), m.simplices)   # the generator's own (host C++) canonical order


@pytest.mark.parametrize("dim", [2, 3])
@pytest.mark.parametrize("n", [1, 31, 2047, 2048, 2049, 8193, 50000])
def test_random_rows_sizes_around_the_segments(dim, n):
    rng = np.random.default_rng(100 * dim + n)
    nV = 300 if n < 3000 else 2**31 - 1   # few ids: many equal columns; huge ids: four passes per column
    S = np.empty((n, dim + 1), dtype=np.int32)
    for i in range(n):   # distinct ids inside a row
        S[i] = rng.choice(nV, size=dim + 1, replace=False) if nV <= 300 else np.unique(rng.integers(0, nV, size=8))[: dim + 1][rng.permutation(dim + 1)]
    _check(dim, nV, S)


def test_duplicated_rows_keep_input_order():
    m = meshgen.make_config(1)
    S = _scramble(np.concatenate([m.simplices, m.simplices[::3], m.simplices[::7]]), 11)
    _check(3, m.num_vertices, S)


def test_empty_and_refusals():
    import torch

    import paper_2507_15230_b200 as gale

    out, perm = gale.canonicalize(3, 10, np.zeros((0, 4), dtype=np.int32))
    assert out.shape == (0, 4) and perm.shape == (0,)
    for bad in ([[0, 1, 2, 2]], [[0, 1, 2, 10]], [[-1, 1, 2, 3]]):
        with pytest.raises(gale.GaleError) as e:
            gale.canonicalize(3, 10, np.array(bad, dtype=np.int32))
        assert e.value.status == gale.ERR_DEGENERATE
    t = torch.zeros((4, 4), dtype=torch.int32, device="cuda")
    with pytest.raises(gale.GaleError) as e:   # aliased input / output
        gale.gale_canonicalize(3, 4, 10, t.data_ptr(), t.data_ptr())
    assert e.value.status == gale.ERR_INVALID_ARG


def test_full_size_config5_scrambled_on_the_device():
    """99.5 M tetrahedra: rows scrambled on the device (seeded), canonicalised, compared with the generator's array."""
    import torch

    import paper_2507_15230_b200 as gale

    m = meshgen.make_config(5)
    T = torch.from_numpy(m.simplices).cuda()
    g = torch.Generator(device="cuda").manual_seed(5)
    order = torch.randperm(T.shape[0], device="cuda", generator=g)
    S = T[order]
    S = torch.stack([S[:, 2], S[:, 0], S[:, 3], S[:, 1]], dim=1).contiguous()   # and the columns rotated
    out, perm = gale.canonicalize(3, m.num_vertices, S)
    assert torch.equal(out, T)
    assert torch.equal(order[perm.long()], torch.arange(T.shape[0], device="cuda"))   # perm undoes the scramble
