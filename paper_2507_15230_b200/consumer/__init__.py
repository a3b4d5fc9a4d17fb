"""Consumers of the relation queue: host threads that pop finished batches from the
pinned result queue and run an analysis on them with a per-vertex scalar field — the paper's consumer
threads — and the waiting-time breakdown the paper reports per request
(enqueue, in-queue, data preparation, kernel + transfer, integration).

The analyses themselves (gale_consumer.cpp, host C++) are Fig. 1's neighbour sum and the
critical-point classification of TTK's CriticalPoints from VV + VT."""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
import time

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gale_consumer.cpp")
_LIB = os.path.join(_HERE, "libgale_consumer.so")
_lib = None
REGULAR, MINIMUM, MAXIMUM, SADDLE = 0, 1, 2, 3


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp, i64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32
        lib.gc_neighbour_sum.restype = None
        lib.gc_neighbour_sum.argtypes = [i64, vp, vp, vp, vp]
        lib.gc_critical_points.restype = None
        lib.gc_critical_points.argtypes = [i64, i32, ctypes.c_int, vp, vp, vp, vp, vp, vp, vp, vp]
        _lib = lib
    return _lib


def _ptr(a):
    return ctypes.c_void_p(a.ctypes.data)


def neighbour_sum(vv_off: np.ndarray, vv_idx: np.ndarray, scalar: np.ndarray) -> np.ndarray:
    """out[r] = sum of scalar over VV(row r) (Fig. 1(c)); rows of one batch or cluster."""
    n = len(vv_off) - 1
    out = np.empty(n, np.float64)
    _load().gc_neighbour_sum(n, _ptr(vv_off), _ptr(vv_idx), _ptr(scalar), _ptr(out))
    return out


def critical_points(first_vertex: int, D: int, vt_off, vt_idx, vv_off, vv_idx, simplices, scalar, counts=None):
    """Type (REGULAR / MINIMUM / MAXIMUM / SADDLE) of the vertices first_vertex .. of one contiguous row range."""
    n = len(vv_off) - 1
    out = np.empty(n, np.uint8)
    _load().gc_critical_points(n, int(first_vertex), D, _ptr(vt_off), _ptr(vt_idx), _ptr(vv_off), _ptr(vv_idx),
                               _ptr(simplices), _ptr(scalar), _ptr(out), _ptr(counts) if counts is not None else None)
    return out


def run_critical_points(mesh, scalar: np.ndarray, *, consumers: int = 4, batch: int = 64, queue_depth: int = 4,
                        kernel_flags: int = 0) -> dict:
    """CriticalPoints over the whole mesh through the producer-consumer queue: one producer thread submits
    every cluster in batches (VV + VT), `consumers` host threads pop finished batches from the pinned queue,
    classify the batch's vertices and release the slot. Returns the class histogram and, per stage of a
    request as the paper breaks it down, the time summed over all batches."""
    import paper_2507_15230_b200 as gale

    _load()
    D = mesh.dim + 1
    T = np.ascontiguousarray(mesh.simplices, np.int32)
    scalar = np.ascontiguousarray(scalar, np.float32)
    gm = gale.GaleMesh(mesh.dim, mesh.num_vertices, T, mesh.cluster_offsets, max_batch_clusters=batch,
                       queue_depth=queue_depth, flags=kernel_flags)
    nC = mesh.num_clusters
    batches = [np.arange(b, min(nC, b + batch), dtype=np.int32) for b in range(0, nC, batch)]
    types = np.zeros(mesh.num_vertices, np.uint8)
    stage = dict(enqueue_ms=0.0, in_queue_ms=0.0, prep_ms=0.0, kernel_ms=0.0, d2h_ms=0.0, integrate_ms=0.0, consume_ms=0.0)
    lock, pop_lock = threading.Lock(), threading.Lock()
    state = dict(submitted=0, done=False, popped=0)

    failed = []                                         # first exception of any thread: everybody stops, the caller gets it

    def guarded(body):
        def run():
            try:
                body()
            except BaseException as e:   # noqa: BLE001 - re-raised in the calling thread after the join
                failed.append(e)
        return run

    def producer():
        for ids in batches:
            t0 = time.perf_counter()
            while gm.compute(ids, gale.REL_VT | gale.REL_VV) == gale.ERR_WOULD_BLOCK:
                if failed:
                    return
                time.sleep(0.0002)                      # bounded queue: back-pressure until a consumer releases
            with lock:
                stage["enqueue_ms"] += 1e3 * (time.perf_counter() - t0)
                state["submitted"] += 1
        state["done"] = True

    def consumer():
        while True:
            if failed:
                return
            with pop_lock:                              # one popping thread at a time (boundary contract)
                if state["done"] and state["popped"] >= len(batches):
                    return
                st, v = gm.pop(20)                      # OK / WOULD_BLOCK / EMPTY; anything else raises (fatal)
                if st == gale.OK:
                    state["popped"] += 1
            if st != gale.OK:
                if state["done"] and state["popped"] >= len(batches):
                    return
                continue
            a = gm.view_arrays(v)
            t0 = time.perf_counter()
            rows = a["vt_row_begin"]
            for i, c in enumerate(a["cluster_ids"]):    # one contiguous vertex range per cluster
                r0, r1 = int(rows[i]), int(rows[i + 1])
                lo = int(mesh.cluster_offsets[c])
                types[lo:lo + (r1 - r0)] = critical_points(lo, D, a["vt_offsets"][r0:r1 + 1], a["vt_indices"],
                                                           a["vv_offsets"][r0:r1 + 1], a["vv_indices"], T, scalar)
            dt = 1e3 * (time.perf_counter() - t0)
            with lock:
                stage["consume_ms"] += dt
                stage["prep_ms"] += v.prep_ms
                stage["kernel_ms"] += v.kernel_ms
                stage["d2h_ms"] += v.d2h_ms
                stage["in_queue_ms"] += max(0.0, v.queue_ms - v.kernel_ms - v.d2h_ms)
            gm.release(v)

    t0 = time.perf_counter()
    th = [threading.Thread(target=guarded(producer))] + [threading.Thread(target=guarded(consumer)) for _ in range(max(1, consumers))]
    for t in th:
        t.start()
    for t in th:
        t.join()
    wall = time.perf_counter() - t0
    info = gm.info
    if failed:
        try:
            gm.destroy()
        finally:
            raise failed[0]
    gm.destroy()
    hist = np.bincount(types, minlength=4)
    return dict(minima=int(hist[MINIMUM]), maxima=int(hist[MAXIMUM]), saddles=int(hist[SADDLE]), regular=int(hist[REGULAR]),
                types=types, wall_s=wall, batches=len(batches), consumers=consumers, stages_ms=stage,
                note="integrate_ms is 0 by construction: the kernels emit global ids, the paper's CPU remap "
                     "(PAPER.md:210, 5.9 % of its run time) does not exist",
                kernel=["dense", "walk"][info.kernel_variant])
