"""gale_canonicalize_static: the canonicalisation entry for callers that cannot allocate device memory.

Some users of this library run where cudaMalloc is not an option: an in-situ analysis loaded into a simulation
whose own pool has claimed the whole GPU (a guest's cudaMalloc fails with out-of-memory there), or a service loop
that must not take the device-wide synchronisation cudaMalloc / cudaFree bring. For them the library offers one
entry whose temporaries live in a fixed array inside the library image (include/gale.h: at most
GALE_CANON_STATIC_MAX_SIMPLICES rows, about 25 MiB per GPU). This file checks that entry against the existing,
allocating gale_canonicalize — integer work, so the bar is the one every parity test here uses: bit-exact —
on two calls in a row, because the array is shared by all calls and keeps the previous call's contents: the
second call (a different mesh, smaller, other dimension) must not see anything of the first, and a refused
(degenerate) call in between must not leave its error flag behind.

The file is named to be collected last (pytest -x stops at the first failure; a failure here must not hide the
parity tests). It holds no state of its own: it passes alone in a fresh process and after the rest of the suite.
"""
import os

import numpy as np
import pytest

import meshgen


def _scramble(T, seed):
    rng = np.random.default_rng(seed)
    rows = T[rng.permutation(len(T))]
    cols = np.argsort(rng.random(rows.shape), axis=1)
    return np.ascontiguousarray(np.take_along_axis(rows, cols, axis=1))


def _same_as_allocating_path(gale, dim, nV, S, want_perm=True):
    """Both entries on the same device input; rows and permutation must agree bit for bit."""
    import torch

    d_in = torch.from_numpy(S).cuda()
    ref, ref_perm = gale.canonicalize(dim, nV, d_in, want_perm=want_perm)
    got, got_perm = gale.canonicalize_static(dim, nV, d_in, want_perm=want_perm)
    assert torch.equal(d_in.cpu(), torch.from_numpy(S))            # the input is not modified
    assert torch.equal(got, ref)
    if want_perm:
        assert torch.equal(got_perm, ref_perm)
    else:
        assert got_perm is None and ref_perm is None
    return got


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_allocating_path():
    import paper_2507_15230_b200 as gale

    # call 1: 3-D, ~214 K rows (105 segments of the radix sort, a ragged last one), duplicated rows included
    big = meshgen.make_mesh(3, 32, clustering="octree", capacity=4096)
    S1 = _scramble(np.concatenate([big.simplices, big.simplices[::5]]), 1)
    out1 = _same_as_allocating_path(gale, 3, big.num_vertices, S1)

    # in between: a refused call (it sets the error flag inside the shared array) ...
    with pytest.raises(gale.GaleError) as e:
        gale.canonicalize_static(3, 10, np.array([[0, 1, 2, 2]], dtype=np.int32))
    assert e.value.status == gale.ERR_DEGENERATE

    # call 2, straight after: other dimension, smaller, no permutation wanted (the library's own buffer in the
    # array is used instead) — whatever calls 1 and the refusal left behind must not show
    small = meshgen.make_delaunay(2, 5000, seed=22, capacity=500)
    S2 = _scramble(small.simplices, 2)
    out2 = _same_as_allocating_path(gale, 2, small.num_vertices, S2, want_perm=False)
    assert np.array_equal(out2.cpu().numpy(), small.simplices)     # = the generator's canonical order

    # and the first input again: same answer as the first time
    out3 = _same_as_allocating_path(gale, 3, big.num_vertices, S1)
    assert np.array_equal(out3.cpu().numpy(), out1.cpu().numpy())


@pytest.mark.gpu
def test_sizes_up_to_the_limit_and_the_empty_list():
    import torch

    import paper_2507_15230_b200 as gale

    out, perm = gale.canonicalize_static(3, 10, np.zeros((0, 4), dtype=np.int32))
    assert out.shape == (0, 4) and perm.shape == (0,)
    # exactly the maximum: random rows built on the device (seeded), ids below 2^20 (three passes per column)
    n, nV = gale.CANON_STATIC_MAX_SIMPLICES, 1 << 20
    g = torch.Generator(device="cuda").manual_seed(7)
    base = torch.randint(0, nV - 3, (n, 1), device="cuda", generator=g, dtype=torch.int32)
    S = (base + torch.tensor([[2, 0, 3, 1]], device="cuda", dtype=torch.int32)).contiguous()   # distinct inside a row
    ref, ref_perm = gale.canonicalize(3, nV, S)
    got, got_perm = gale.canonicalize_static(3, nV, S)
    assert torch.equal(got, ref) and torch.equal(got_perm, ref_perm)


def test_rows_beyond_the_limit_are_refused_before_anything_runs():
    """Needs no GPU: the size is checked before any pointer or device is touched."""
    import paper_2507_15230_b200 as gale

    gale.load_library(build_if_missing=True)
    with pytest.raises(gale.GaleError) as e:
        gale.gale_canonicalize_static(3, gale.CANON_STATIC_MAX_SIMPLICES + 1, 100, 256, 512, 0, 0)
    assert e.value.status == gale.ERR_WORKSPACE
    assert "GALE_CANON_STATIC_MAX_SIMPLICES" in str(e.value)
    hdr = open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", "include", "gale.h")).read()
    assert "#define GALE_CANON_STATIC_MAX_SIMPLICES (1 << 20)" in hdr   # the binding's constant is the header's
