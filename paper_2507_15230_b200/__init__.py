"""paper_2507_15230_b200 — Python binding of the B200-native GALE relation hot path.

Thin ctypes marshalling over the C ABI in include/gale.h (csrc/libgale.so): every relation entry is
computed by the CUDA kernels in csrc/gale_kernels.cuh. PyTorch only provides device memory and
streams. There is no CPU fallback: if libgale.so is missing or no sm_100 device is present the calls
raise GaleError.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from .build import LIB, build_library

REL_VT, REL_VV, REL_TT, REL_ALL = 1, 2, 4, 7
REL_VE, REL_VF = 8, 16
REL_EF, REL_ET, REL_FT = 32, 64, 128
VALIDATE, VALIDATE_MANIFOLD, STREAM_ORDERED, KERNEL_DENSE, KERNEL_WALK, STAGE_FROM_T = 1, 2, 4, 8, 16, 32
WITH_EDGES, WITH_FACETS, WITH_COBOUNDARY = 64, 128, 256
OK, ERR_INVALID_ARG, ERR_NOT_CANONICAL, ERR_DEGENERATE, ERR_NONMANIFOLD, ERR_BAD_CLUSTER = 0, -1, -2, -3, -4, -5
ERR_WOULD_BLOCK, ERR_EMPTY, ERR_WORKSPACE, ERR_CUDA, ERR_UNSUPPORTED = -6, -7, -8, -9, -10

_i32p = ctypes.POINTER(ctypes.c_int32)


class gale_mesh_desc_t(ctypes.Structure):
    _fields_ = [("dim", ctypes.c_int32), ("num_vertices", ctypes.c_int32), ("num_simplices", ctypes.c_int64),
                ("d_simplices", ctypes.c_void_p), ("num_clusters", ctypes.c_int32),
                ("h_cluster_offsets", _i32p), ("max_batch_clusters", ctypes.c_int32),
                ("queue_depth", ctypes.c_int32), ("device_ring", ctypes.c_int32), ("tile_vertices", ctypes.c_int32),
                ("d_workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t), ("flags", ctypes.c_uint32)]


class gale_batch_view_t(ctypes.Structure):
    _fields_ = [("sequence", ctypes.c_int64), ("n_clusters", ctypes.c_int32), ("relation_mask", ctypes.c_uint32),
                ("dim", ctypes.c_int32), ("on_device", ctypes.c_int32),
                ("cluster_ids", _i32p), ("vt_row_begin", _i32p), ("tt_row_begin", _i32p),
                ("vt_rows", ctypes.c_int64), ("vt_nnz", ctypes.c_int64),
                ("vt_offsets", ctypes.c_void_p), ("vt_indices", ctypes.c_void_p),
                ("vv_rows", ctypes.c_int64), ("vv_nnz", ctypes.c_int64),
                ("vv_offsets", ctypes.c_void_p), ("vv_indices", ctypes.c_void_p),
                ("tt_rows", ctypes.c_int64), ("tt_indices", ctypes.c_void_p),
                ("kernel_ms", ctypes.c_float), ("slot", ctypes.c_int32),
                ("prep_ms", ctypes.c_float), ("d2h_ms", ctypes.c_float), ("queue_ms", ctypes.c_float),
                ("reserved", ctypes.c_int32),
                ("ve_indices", ctypes.c_void_p), ("vf_nnz", ctypes.c_int64),
                ("vf_offsets", ctypes.c_void_p), ("vf_indices", ctypes.c_void_p),
                ("e_row_begin", _i32p), ("f_row_begin", _i32p),
                ("ef_nnz", ctypes.c_int64), ("et_nnz", ctypes.c_int64), ("ft_nnz", ctypes.c_int64),
                ("ef_offsets", ctypes.c_void_p), ("ef_indices", ctypes.c_void_p),
                ("et_offsets", ctypes.c_void_p), ("et_indices", ctypes.c_void_p),
                ("ft_offsets", ctypes.c_void_p), ("ft_indices", ctypes.c_void_p)]


class gale_mesh_info_t(ctypes.Structure):
    _fields_ = [("tile_vertices", ctypes.c_int32), ("num_tiles", ctypes.c_int32),
                ("num_external_refs", ctypes.c_int64), ("vt_nnz", ctypes.c_int64), ("vv_nnz", ctypes.c_int64),
                ("smem_bytes", ctypes.c_int32), ("max_staged", ctypes.c_int32),
                ("slot_bytes", ctypes.c_size_t), ("workspace_used", ctypes.c_size_t), ("create_ms", ctypes.c_double),
                ("local_id_bytes", ctypes.c_int32), ("block_threads", ctypes.c_int32),
                ("index_bytes", ctypes.c_size_t), ("num_edges", ctypes.c_int64), ("num_triangles", ctypes.c_int64),
                ("kernel_variant", ctypes.c_int32),
                ("tune_dense_ms", ctypes.c_float), ("tune_walk_ms", ctypes.c_float), ("reserved", ctypes.c_int32)]


class gale_tile_view_t(ctypes.Structure):
    _fields_ = [("v_lo", ctypes.c_int32), ("nrows", ctypes.c_int32), ("t_lo", ctypes.c_int32),
                ("num_internal", ctypes.c_int32), ("num_external", ctypes.c_int32),
                ("num_lower_halo", ctypes.c_int32), ("num_local", ctypes.c_int32), ("cluster", ctypes.c_int32),
                ("d_external", ctypes.c_void_p), ("d_local_to_global", ctypes.c_void_p)]


EXPORTS = ["gale_canonicalize", "gale_canonicalize_static", "gale_boundary_lookup", "gale_mesh_edges", "gale_mesh_triangles", "gale_mesh_tile", "gale_mesh_interval_array", "gale_plan_create", "gale_plan_workspace_bytes", "gale_plan_destroy", "gale_mesh_create_planned",
           "gale_mesh_workspace_bytes", "gale_mesh_create", "gale_mesh_info", "gale_cluster_batch_compute",
           "gale_queue_pop", "gale_queue_release", "gale_destroy", "gale_status_string", "gale_last_error"]


class GaleError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        super().__init__(f"{where}: {status_string(status)} ({status}) {detail}".rstrip())


_lib = None


def load_library(build_if_missing: bool = False) -> ctypes.CDLL:
    """dlopen csrc/libgale.so (fails loudly when it was not built: there is no fallback path)."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing:
        build_library()
    path = os.environ.get("GALE_LIBRARY", LIB)   # another build of the same sources, e.g. libgale_checked.so
    if not os.path.exists(path):
        raise RuntimeError(f"{path} not built (no fallback path exists); run "
                           "`python -c 'import __graft_entry__ as g; g.build()'`")
    lib = ctypes.CDLL(path)
    vp = ctypes.c_void_p
    lib.gale_canonicalize.restype = ctypes.c_int32
    lib.gale_canonicalize.argtypes = [ctypes.c_int32, ctypes.c_int64, ctypes.c_int32, vp, vp, vp, vp]
    lib.gale_canonicalize_static.restype = ctypes.c_int32
    lib.gale_canonicalize_static.argtypes = [ctypes.c_int32, ctypes.c_int64, ctypes.c_int32, vp, vp, vp, vp]
    lib.gale_boundary_lookup.restype = ctypes.c_int32
    lib.gale_boundary_lookup.argtypes = [vp, ctypes.c_int32, ctypes.c_int64, ctypes.c_int64, vp, vp]
    lib.gale_plan_create.restype = ctypes.c_int32
    lib.gale_plan_create.argtypes = [ctypes.POINTER(gale_mesh_desc_t), vp, ctypes.POINTER(vp)]
    lib.gale_plan_workspace_bytes.restype = ctypes.c_int32
    lib.gale_plan_workspace_bytes.argtypes = [vp, ctypes.POINTER(ctypes.c_size_t)]
    lib.gale_plan_destroy.restype = ctypes.c_int32
    lib.gale_plan_destroy.argtypes = [vp]
    lib.gale_mesh_create_planned.restype = ctypes.c_int32
    lib.gale_mesh_create_planned.argtypes = [vp, vp, ctypes.c_size_t, vp, ctypes.POINTER(vp)]
    lib.gale_mesh_workspace_bytes.restype = ctypes.c_int32
    lib.gale_mesh_workspace_bytes.argtypes = [ctypes.POINTER(gale_mesh_desc_t), vp, ctypes.POINTER(ctypes.c_size_t)]
    lib.gale_mesh_create.restype = ctypes.c_int32
    lib.gale_mesh_create.argtypes = [ctypes.POINTER(gale_mesh_desc_t), vp, ctypes.POINTER(vp)]
    lib.gale_mesh_info.restype = ctypes.c_int32
    lib.gale_mesh_info.argtypes = [vp, ctypes.POINTER(gale_mesh_info_t)]
    lib.gale_mesh_edges.restype = ctypes.c_int32
    lib.gale_mesh_edges.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(ctypes.c_int64)]
    lib.gale_mesh_triangles.restype = ctypes.c_int32
    lib.gale_mesh_triangles.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(ctypes.c_int64)]
    lib.gale_mesh_tile.restype = ctypes.c_int32
    lib.gale_mesh_tile.argtypes = [vp, ctypes.c_int32, ctypes.POINTER(gale_tile_view_t)]
    lib.gale_mesh_interval_array.restype = ctypes.c_int32
    lib.gale_mesh_interval_array.argtypes = [vp, ctypes.POINTER(vp)]
    lib.gale_cluster_batch_compute.restype = ctypes.c_int32
    lib.gale_cluster_batch_compute.argtypes = [vp, ctypes.c_uint32, _i32p, ctypes.c_int32, vp]
    lib.gale_queue_pop.restype = ctypes.c_int32
    lib.gale_queue_pop.argtypes = [vp, ctypes.POINTER(gale_batch_view_t), ctypes.c_int32]
    lib.gale_queue_release.restype = ctypes.c_int32
    lib.gale_queue_release.argtypes = [vp, ctypes.POINTER(gale_batch_view_t)]
    lib.gale_destroy.restype = ctypes.c_int32
    lib.gale_destroy.argtypes = [vp]
    lib.gale_status_string.restype = ctypes.c_char_p
    lib.gale_status_string.argtypes = [ctypes.c_int32]
    lib.gale_last_error.restype = ctypes.c_char_p
    lib.gale_last_error.argtypes = []
    _lib = lib
    return lib


def status_string(status: int) -> str:
    return load_library().gale_status_string(int(status)).decode()


def _check(status: int, where: str):
    if status != OK:
        raise GaleError(status, where, load_library().gale_last_error().decode())


# ---- the C-ABI calls, same names, marshalling only ----------------------------------------------------
def gale_canonicalize(dim: int, num_simplices: int, num_vertices: int, d_in: int, d_out: int, d_perm: int = 0,
                      cuda_stream: int = 0) -> None:
    """DEVICE pointers in, DEVICE pointers out (include/gale.h); d_perm = 0 skips the permutation."""
    _check(load_library().gale_canonicalize(dim, num_simplices, num_vertices, ctypes.c_void_p(d_in), ctypes.c_void_p(d_out),
                                            ctypes.c_void_p(d_perm or None), ctypes.c_void_p(cuda_stream)), "gale_canonicalize")


def canonicalize(dim: int, num_vertices: int, simplices, want_perm: bool = True):
    """Argument marshalling for gale_canonicalize: `simplices` is a CUDA int32 tensor [n, dim+1] (or anything
    torch.as_tensor takes, uploaded first); returns (canonical simplices, permutation or None) as CUDA tensors."""
    import torch

    t = torch.as_tensor(simplices, dtype=torch.int32)
    if t.device.type != "cuda":
        t = t.cuda()
    t = t.contiguous().reshape(-1, dim + 1)
    out = torch.empty_like(t)
    perm = torch.empty(t.shape[0], dtype=torch.int32, device=t.device) if want_perm else None
    gale_canonicalize(dim, t.shape[0], num_vertices, t.data_ptr(), out.data_ptr(), perm.data_ptr() if want_perm else 0,
                      torch.cuda.current_stream().cuda_stream)
    return out, perm


CANON_STATIC_MAX_SIMPLICES = 1 << 20   # GALE_CANON_STATIC_MAX_SIMPLICES of include/gale.h


def gale_canonicalize_static(dim: int, num_simplices: int, num_vertices: int, d_in: int, d_out: int, d_perm: int = 0,
                             cuda_stream: int = 0) -> None:
    """gale_canonicalize for callers that may not allocate device memory (include/gale.h): the library makes no
    cudaMalloc / cudaFree here, its temporaries sit in a fixed array inside the library image, which limits the
    call to CANON_STATIC_MAX_SIMPLICES rows (ERR_WORKSPACE beyond). Same pointers, results and errors otherwise."""
    _check(load_library().gale_canonicalize_static(dim, num_simplices, num_vertices, ctypes.c_void_p(d_in), ctypes.c_void_p(d_out),
                                                   ctypes.c_void_p(d_perm or None), ctypes.c_void_p(cuda_stream)),
           "gale_canonicalize_static")


def canonicalize_static(dim: int, num_vertices: int, simplices, want_perm: bool = True):
    """Argument marshalling for gale_canonicalize_static, same shape as `canonicalize`. Note that this helper itself
    creates the output tensors with torch (the caller's side of the contract: inputs and outputs are the caller's);
    a caller that really cannot allocate passes pointers it already owns to gale_canonicalize_static directly."""
    import torch

    t = torch.as_tensor(simplices, dtype=torch.int32)
    if t.device.type != "cuda":
        t = t.cuda()
    t = t.contiguous().reshape(-1, dim + 1)
    out = torch.empty_like(t)
    perm = torch.empty(t.shape[0], dtype=torch.int32, device=t.device) if want_perm else None
    gale_canonicalize_static(dim, t.shape[0], num_vertices, t.data_ptr(), out.data_ptr(), perm.data_ptr() if want_perm else 0,
                             torch.cuda.current_stream().cuda_stream)
    return out, perm


BND_FE, BND_TE, BND_TF = 1, 2, 3


def gale_boundary_lookup(handle, relation: int, first_id: int, count: int, d_out: int, cuda_stream: int = 0) -> None:
    _check(load_library().gale_boundary_lookup(handle, relation, first_id, count, ctypes.c_void_p(d_out or None),
                                               ctypes.c_void_p(cuda_stream)), "gale_boundary_lookup")


def gale_plan_create(desc: gale_mesh_desc_t, cuda_stream: int = 0) -> ctypes.c_void_p:
    h = ctypes.c_void_p()
    _check(load_library().gale_plan_create(ctypes.byref(desc), ctypes.c_void_p(cuda_stream), ctypes.byref(h)),
           "gale_plan_create")
    return h


def gale_plan_workspace_bytes(plan) -> int:
    out = ctypes.c_size_t(0)
    _check(load_library().gale_plan_workspace_bytes(plan, ctypes.byref(out)), "gale_plan_workspace_bytes")
    return int(out.value)


def gale_plan_destroy(plan) -> None:
    _check(load_library().gale_plan_destroy(plan), "gale_plan_destroy")


def gale_mesh_create_planned(plan, d_workspace: int, workspace_bytes: int, cuda_stream: int = 0) -> ctypes.c_void_p:
    h = ctypes.c_void_p()
    _check(load_library().gale_mesh_create_planned(plan, ctypes.c_void_p(d_workspace), workspace_bytes,
                                                   ctypes.c_void_p(cuda_stream), ctypes.byref(h)),
           "gale_mesh_create_planned")
    return h


def gale_mesh_workspace_bytes(desc: gale_mesh_desc_t, cuda_stream: int = 0) -> int:
    out = ctypes.c_size_t(0)
    _check(load_library().gale_mesh_workspace_bytes(ctypes.byref(desc), ctypes.c_void_p(cuda_stream), ctypes.byref(out)),
           "gale_mesh_workspace_bytes")
    return int(out.value)


def gale_mesh_create(desc: gale_mesh_desc_t, cuda_stream: int = 0) -> ctypes.c_void_p:
    h = ctypes.c_void_p()
    _check(load_library().gale_mesh_create(ctypes.byref(desc), ctypes.c_void_p(cuda_stream), ctypes.byref(h)),
           "gale_mesh_create")
    return h


def gale_mesh_info(handle) -> gale_mesh_info_t:
    info = gale_mesh_info_t()
    _check(load_library().gale_mesh_info(handle, ctypes.byref(info)), "gale_mesh_info")
    return info


def _sub_list(fn, handle, where):
    first, other, n = ctypes.c_void_p(), ctypes.c_void_p(), ctypes.c_int64()
    _check(fn(handle, ctypes.byref(first), ctypes.byref(other), ctypes.byref(n)), where)
    return int(first.value), int(other.value or 0), int(n.value)


def gale_mesh_edges(handle):
    """(DEVICE address of I_E per vertex, DEVICE address of the edges' upper vertices, number of edges)."""
    return _sub_list(load_library().gale_mesh_edges, handle, "gale_mesh_edges")


def gale_mesh_triangles(handle):
    """(DEVICE address of I_F per vertex, DEVICE address of (second, third) vertex pairs, number of triangles)."""
    return _sub_list(load_library().gale_mesh_triangles, handle, "gale_mesh_triangles")


def gale_mesh_tile(handle, tile: int) -> gale_tile_view_t:
    v = gale_tile_view_t()
    _check(load_library().gale_mesh_tile(handle, tile, ctypes.byref(v)), "gale_mesh_tile")
    return v


def gale_mesh_interval_array(handle) -> int:
    """DEVICE address of I_T per vertex (int32[num_vertices + 1])."""
    ptr = ctypes.c_void_p()
    _check(load_library().gale_mesh_interval_array(handle, ctypes.byref(ptr)), "gale_mesh_interval_array")
    return int(ptr.value)


def gale_cluster_batch_compute(handle, relation_mask: int, cluster_ids, cuda_stream: int = 0) -> int:
    """Returns the status (OK or ERR_WOULD_BLOCK); other errors raise."""
    ids = np.ascontiguousarray(cluster_ids, dtype=np.int32)
    st = load_library().gale_cluster_batch_compute(handle, relation_mask, ids.ctypes.data_as(_i32p), len(ids),
                                                   ctypes.c_void_p(cuda_stream))
    if st not in (OK, ERR_WOULD_BLOCK):
        _check(st, "gale_cluster_batch_compute")
    return st


def gale_queue_pop(handle, timeout_ms: int = -1):
    """Returns (status, view); status is OK, ERR_EMPTY or ERR_WOULD_BLOCK; other errors raise. ERR_WORKSPACE (a device
    capacity guard fired, include/gale.h) still pops the batch: its slot is given back here before raising."""
    view = gale_batch_view_t()
    lib = load_library()
    st = lib.gale_queue_pop(handle, ctypes.byref(view), timeout_ms)
    if st not in (OK, ERR_EMPTY, ERR_WOULD_BLOCK):
        detail = lib.gale_last_error().decode()
        if st == ERR_WORKSPACE:
            lib.gale_queue_release(handle, ctypes.byref(view))
        raise GaleError(st, "gale_queue_pop", detail)
    return st, view


def gale_queue_release(handle, view: gale_batch_view_t) -> None:
    _check(load_library().gale_queue_release(handle, ctypes.byref(view)), "gale_queue_release")


def gale_destroy(handle) -> None:
    _check(load_library().gale_destroy(handle), "gale_destroy")


# ---- convenience holder (keeps the torch tensors alive; still marshalling only) ----------------------
class GaleMesh:
    """Owns the device tensors (simplices, workspace) behind one gale_mesh_t handle."""

    def __init__(self, dim: int, num_vertices: int, simplices, cluster_offsets, *, max_batch_clusters: int = 64,
                 queue_depth: int = 0, device_ring: int = 0, tile_vertices: int = 0, flags: int = VALIDATE,
                 device="cuda:0"):
        import torch

        load_library()
        if not torch.cuda.is_available():
            raise GaleError(ERR_UNSUPPORTED, "GaleMesh", "no CUDA device (there is no CPU fallback)")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        if isinstance(simplices, torch.Tensor):
            self.simplices = simplices.to(device=self.device, dtype=torch.int32).contiguous()
        else:
            self.simplices = torch.from_numpy(np.ascontiguousarray(simplices, dtype=np.int32)).to(self.device)
        self.dim, self.D = dim, dim + 1
        self.offsets = np.ascontiguousarray(cluster_offsets, dtype=np.int32)
        d = gale_mesh_desc_t()
        d.dim, d.num_vertices, d.num_simplices = dim, int(num_vertices), int(self.simplices.shape[0])
        d.d_simplices = self.simplices.data_ptr() if d.num_simplices else None
        d.num_clusters = len(self.offsets) - 1
        d.h_cluster_offsets = self.offsets.ctypes.data_as(_i32p)
        d.max_batch_clusters, d.queue_depth, d.device_ring = max_batch_clusters, queue_depth, device_ring
        d.tile_vertices, d.flags = tile_vertices, flags
        self.desc = d
        stream = torch.cuda.current_stream(self.device).cuda_stream
        plan = gale_plan_create(d, stream)                 # the initialization analysis, once
        try:
            nbytes = gale_plan_workspace_bytes(plan)
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            d.d_workspace, d.workspace_bytes = self.workspace.data_ptr(), nbytes
            self.handle = gale_mesh_create_planned(plan, self.workspace.data_ptr(), nbytes, stream)
        finally:
            gale_plan_destroy(plan)
        self.info = gale_mesh_info(self.handle)

    def device_array(self, ptr: int, n: int):
        """int32 torch view of n entries of the workspace at DEVICE address ptr (index arrays, slots)."""
        if not ptr or n == 0:
            return self.torch.empty(0, dtype=self.torch.int32, device=self.device)
        off = ptr - self.workspace.data_ptr()
        return self.workspace[off:off + 4 * n].view(self.torch.int32)

    def compute(self, cluster_ids, relation_mask: int = REL_ALL, stream=None) -> int:
        s = (stream or self.torch.cuda.current_stream(self.device)).cuda_stream
        return gale_cluster_batch_compute(self.handle, relation_mask, cluster_ids, s)

    def pop(self, timeout_ms: int = -1):
        return gale_queue_pop(self.handle, timeout_ms)

    def release(self, view) -> None:
        gale_queue_release(self.handle, view)

    def _array(self, view, ptr, n):
        """int32 array over slot memory: a torch view of the workspace (device) or numpy (pinned host)."""
        if not ptr or n == 0:
            return self.torch.empty(0, dtype=self.torch.int32, device=self.device) if view.on_device else np.empty(0, np.int32)
        if view.on_device:
            off = ptr - self.workspace.data_ptr()
            return self.workspace[off:off + 4 * n].view(self.torch.int32)
        return np.ctypeslib.as_array(ctypes.cast(ptr, _i32p), shape=(n,))

    def view_arrays(self, view) -> dict:
        """Expose a popped view as arrays (no copies of the slot data)."""
        n = view.n_clusters
        out = dict(sequence=view.sequence, n_clusters=n, relation_mask=view.relation_mask, kernel_ms=view.kernel_ms,
                   prep_ms=view.prep_ms, d2h_ms=view.d2h_ms, queue_ms=view.queue_ms,
                   cluster_ids=np.ctypeslib.as_array(view.cluster_ids, shape=(n,)).copy() if n else np.empty(0, np.int32),
                   vt_row_begin=np.ctypeslib.as_array(view.vt_row_begin, shape=(n + 1,)).copy(),
                   tt_row_begin=np.ctypeslib.as_array(view.tt_row_begin, shape=(n + 1,)).copy())
        if view.relation_mask & REL_VT:
            out["vt_offsets"] = self._array(view, view.vt_offsets, view.vt_rows + 1)
            out["vt_indices"] = self._array(view, view.vt_indices, view.vt_nnz)
        if view.relation_mask & REL_VV:
            out["vv_offsets"] = self._array(view, view.vv_offsets, view.vv_rows + 1)
            out["vv_indices"] = self._array(view, view.vv_indices, view.vv_nnz)
        if view.relation_mask & REL_TT:
            out["tt_indices"] = self._array(view, view.tt_indices, view.tt_rows * self.D)
        if view.relation_mask & REL_VE:
            out["ve_indices"] = self._array(view, view.ve_indices, view.vv_nnz)
        if view.relation_mask & REL_VF:
            out["vf_offsets"] = self._array(view, view.vf_offsets, int(out["vt_row_begin"][-1]) + 1)
            out["vf_indices"] = self._array(view, view.vf_indices, view.vf_nnz)
        if view.relation_mask & (REL_EF | REL_ET | REL_FT):
            out["e_row_begin"] = np.ctypeslib.as_array(view.e_row_begin, shape=(n + 1,)).copy()
            out["f_row_begin"] = np.ctypeslib.as_array(view.f_row_begin, shape=(n + 1,)).copy()
            for key, bit, rb in (("ef", REL_EF, "e_row_begin"), ("et", REL_ET, "e_row_begin"), ("ft", REL_FT, "f_row_begin")):
                if view.relation_mask & bit:
                    out[key + "_offsets"] = self._array(view, getattr(view, key + "_offsets"), int(out[rb][-1]) + 1)
                    out[key + "_indices"] = self._array(view, getattr(view, key + "_indices"), getattr(view, key + "_nnz"))
        return out

    def run_batch(self, cluster_ids, relation_mask: int = REL_ALL) -> dict:
        """compute + pop + copy to host numpy + release (test helper; the arithmetic is all on the GPU)."""
        st = self.compute(cluster_ids, relation_mask)
        if st != OK:
            raise GaleError(st, "run_batch")
        st, view = self.pop(-1)
        if st != OK:
            raise GaleError(st, "run_batch/pop")
        arr = self.view_arrays(view)
        host = {}
        for k, v in arr.items():
            if hasattr(v, "cpu"):
                host[k] = v.cpu().numpy()
            elif isinstance(v, np.ndarray):
                host[k] = np.array(v, copy=True)
            else:
                host[k] = v
        self.release(view)
        return host

    def boundary(self, relation: int, first_id: int, count: int):
        """FE / TE / TF rows [first_id, first_id + count) as a CUDA int32 tensor [count, width] (marshalling only)."""
        import torch

        width = 4 if relation == BND_TF else (3 if relation == BND_FE or self.dim == 2 else 6)
        out = torch.empty((count, width), dtype=torch.int32, device="cuda")
        gale_boundary_lookup(self.handle, relation, first_id, count, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
        return out

    def destroy(self) -> None:
        if getattr(self, "handle", None):
            gale_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def split_batch(host: dict, D: int) -> list:
    """Cut a host copy of a batch (run_batch) into per-cluster CSR pieces, offsets restarted at 0."""
    res = []
    for i in range(host["n_clusters"]):
        r0, r1 = int(host["vt_row_begin"][i]), int(host["vt_row_begin"][i + 1])
        t0, t1 = int(host["tt_row_begin"][i]), int(host["tt_row_begin"][i + 1])
        item = dict(cluster=int(host["cluster_ids"][i]))
        for k in ("vt", "vv", "vf"):
            if k + "_offsets" in host:
                off = host[k + "_offsets"][r0:r1 + 1]
                item[k] = ((off - off[0]).astype(np.int32), host[k + "_indices"][off[0]:off[-1]])
        if "ve_indices" in host:                          # VE shares the rows and offsets of VV
            off = host["vv_offsets"][r0:r1 + 1]
            item["ve"] = ((off - off[0]).astype(np.int32), host["ve_indices"][off[0]:off[-1]])
        if "tt_indices" in host:
            item["tt"] = host["tt_indices"][t0 * D:t1 * D].reshape(-1, D)
        for k, rb in (("ef", "e_row_begin"), ("et", "e_row_begin"), ("ft", "f_row_begin")):
            if k + "_offsets" in host:                    # rows = the cluster's own edges / triangles
                q0, q1 = int(host[rb][i]), int(host[rb][i + 1])
                off = host[k + "_offsets"][q0:q1 + 1]
                item[k] = ((off - off[0]).astype(np.int32), host[k + "_indices"][off[0]:off[-1]])
        res.append(item)
    return res
