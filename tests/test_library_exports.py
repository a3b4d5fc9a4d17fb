"""CPU-only: the C-ABI library builds/loads and exports every symbol include/gale.h declares;
the Python binding mirrors the header's structs. No compute call is made here."""
import ctypes
import os
import re

import pytest

import paper_2507_15230_b200 as gale

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    return gale.load_library(build_if_missing=True)


def _declared():
    src = open(os.path.join(ROOT, "include", "gale.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gale_[a-z_]+)\s*\(", src)))


def test_exports_every_declared_symbol(lib):
    names = _declared()
    assert {"gale_mesh_create", "gale_cluster_batch_compute", "gale_queue_pop", "gale_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(gale.EXPORTS) == names


def test_status_strings(lib):
    assert gale.status_string(0) == "GALE_OK"
    assert gale.status_string(gale.ERR_WOULD_BLOCK) == "GALE_ERR_WOULD_BLOCK"
    assert gale.status_string(-99) == "GALE_ERR_UNKNOWN"


def test_struct_layout_matches_header():
    # sizes implied by include/gale.h on LP64
    assert ctypes.sizeof(gale.gale_mesh_desc_t) == 80
    assert ctypes.sizeof(gale.gale_batch_view_t) == 272
    assert ctypes.sizeof(gale.gale_mesh_info_t) == 112      # gcc sizeof(gale_mesh_info_t) of include/gale.h


def test_argument_errors_without_gpu(lib):
    # null / malformed descriptors are refused before any CUDA call
    out = ctypes.c_size_t()
    assert lib.gale_mesh_workspace_bytes(None, None, ctypes.byref(out)) == gale.ERR_INVALID_ARG
    d = gale.gale_mesh_desc_t()
    d.dim = 5
    assert lib.gale_mesh_workspace_bytes(ctypes.byref(d), None, ctypes.byref(out)) == gale.ERR_INVALID_ARG
    assert lib.gale_destroy(None) == gale.ERR_INVALID_ARG
    assert lib.gale_queue_pop(None, None, 0) == gale.ERR_INVALID_ARG
    # GALE_STAGE_FROM_T selects the dense kernel; asking for the walk kernel as well is a contradiction
    import numpy as np
    off = np.array([0, 5], np.int32)
    d = gale.gale_mesh_desc_t()
    d.dim, d.num_vertices, d.num_simplices, d.num_clusters, d.max_batch_clusters = 3, 5, 0, 1, 1
    d.h_cluster_offsets = off.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))
    d.flags = gale.STAGE_FROM_T | gale.KERNEL_WALK
    assert lib.gale_mesh_workspace_bytes(ctypes.byref(d), None, ctypes.byref(out)) == gale.ERR_INVALID_ARG


def test_no_cpu_fallback(lib):
    """Without a CUDA device the product path must fail loudly (never route through a CPU path)."""
    import numpy as np
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    off = np.array([0, 5], np.int32)
    d = gale.gale_mesh_desc_t()
    d.dim, d.num_vertices, d.num_simplices, d.num_clusters = 3, 5, 0, 1
    d.h_cluster_offsets = off.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))
    d.max_batch_clusters = 1
    with pytest.raises(gale.GaleError) as e:
        gale.gale_mesh_workspace_bytes(d)
    assert e.value.status == gale.ERR_UNSUPPORTED
    with pytest.raises(gale.GaleError):
        gale.GaleMesh(3, 5, np.zeros((0, 4), np.int32), off)
