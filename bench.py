#!/usr/bin/env python
"""bench.py — tets/s through VT+VV+TT per cluster batch, and the HBM roofline fraction.

A *step* is one pass of the whole hot path over the whole mesh: every
cluster once, in batches of `--batch` clusters (config 5: 4,096 clusters -> 64 batches of 64), results
kept in the device ring (queue_depth = 0). `value` = simplices / device time of a step.
`e2e` is the same pass through the C ABI with HOST buffers: the simplex array is copied from pinned
host memory each step and every batch is streamed D2H through the pinned result queue (a7) and
popped/released on the host.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--n GRID] [--impl reference]

Under torchrun (N > 1) every rank runs an independent replica of the same pass (the path has no
exchange step: clusters are independent); rank 0 prints the one JSON line.
"""
from __future__ import annotations

import argparse
import collections
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import meshgen  # noqa: E402

METRIC = "tets/s through VT+VV+TT per cluster batch"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback


def algorithmic_bytes(dim, n_simplices, rows, vt_nnz, vv_nnz, tt_rows, n_batches):
    """Compulsory bytes of a pass: each simplex row read once, each output
    array written once (indices + offsets)."""
    D = dim + 1
    return 4 * D * n_simplices + 4 * (vt_nnz + vv_nnz) + 4 * D * tt_rows + 2 * 4 * (rows + n_batches)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        sel = [r for (t, r) in self.rows if t0 <= t <= t1] or [r for (_, r) in self.rows[-3:]]
        sm, mx, reasons = [], [], set()
        for r in sel:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def max_over_ranks(x: float, dist=None, device="cuda") -> float:
    """Timing rule of the bench contract: a multi-rank number is the MAX over ranks (the slowest replica).
    `dist` is torch.distributed when WORLD_SIZE > 1, else None."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, units_per_rank: int, ms_per_step: float) -> float:
    """`value` of the JSON line: units processed by ALL ranks (independent replicas: the path has no
    exchange step) divided by the max-over-ranks time of a step."""
    return world * units_per_rank / (ms_per_step * 1e-3)


def make_workload(args):
    t0 = time.time()
    mesh = meshgen.make_config(args.config, n=args.n)
    return mesh, time.time() - t0


def oracle_sample(mesh, target_s=15.0, max_clusters=256, clusters=None):
    """Time the CPU oracle (as it stands, single thread, pinned to ONE host core) on a bounded sample of the
    same mesh: whole clusters spread over the mesh, restricted evaluation (oracle/gale_oracle.cpp), one call
    whose cluster count is calibrated to about target_s seconds of relation work.

    The restricted oracle first cuts the sub-mesh of the selection out of the whole mesh (two scans over
    all simplices, a fixed cost per call that says nothing about the relations); the oracle's own timers
    separate it, so the rate is  internal simplices of the sample / (VT + VV + TT seconds)  and both
    bench arms (--impl reference, cpu_baseline) report the same quantity. Returns a dict."""
    import oracle

    first = np.searchsorted(mesh.simplices[:, 0], mesh.cluster_offsets)
    nC = mesh.num_clusters
    core = None
    old_aff = None
    try:
        old_aff = os.sched_getaffinity(0)
        core = sorted(old_aff)[len(old_aff) // 2]
        os.sched_setaffinity(0, {core})
    except (AttributeError, OSError):
        pass

    def run(k):
        sel = np.linspace(0, nC - 1, num=k).astype(int).tolist() if k < nC else list(range(nC))
        t0 = time.perf_counter()
        oracle.cluster_results(mesh.dim, mesh.num_vertices, mesh.simplices, mesh.cluster_offsets, sel, restricted=True)
        wall = time.perf_counter() - t0
        return wall, int(sum(first[c + 1] - first[c] for c in set(sel))), dict(oracle.last_timing)

    try:
        k = min(nC, clusters or 4)      # `clusters`: a count calibrated by an earlier call (no second run)
        wall, done, tm = run(k)
        rel = tm["vt"] + tm["vv"] + tm["tt"]
        if clusters is None and rel < target_s / 2 and k < min(nC, max_clusters):
            k = int(max(k, min(nC, max_clusters, k * target_s / max(rel, 1e-6))))
            wall, done, tm = run(k)
            rel = tm["vt"] + tm["vv"] + tm["tt"]
    finally:
        if old_aff is not None:
            try:
                os.sched_setaffinity(0, old_aff)
            except OSError:
                pass
    rel = max(rel, 1e-9)
    return {"value": done / rel, "clusters": k, "internal_simplices": done, "sub_mesh_simplices": tm["sub_simplices"],
            "relation_s": rel, "extract_s": tm["extract"], "wall_s": wall, "pinned_core": core,
            "per_relation_tets_per_s": {"VT": done / max(tm["vt"], 1e-9), "VV": done / max(tm["vv"], 1e-9),
                                        "TT": done / max(tm["tt"], 1e-9)},
            "sample": (f"{k} whole clusters spread over the same mesh ({done} internal simplices; the restricted oracle "
                       f"evaluates the definitions on their {tm['sub_simplices']}-simplex closure), VT+VV+TT {rel:.2f} s on "
                       f"core {core}; cutting the closure out of the whole mesh took {tm['extract']:.2f} s more and is "
                       f"not counted")}


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    mesh, _ = make_workload(args)
    n = max(1, args.steps + args.warmup)
    per_step = max(1.0, min(15.0, 100.0 / n))       # seconds of relation work per step
    vals, secs, last = [], [], None
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        last = oracle_sample(mesh, target_s=per_step, max_clusters=256, clusters=last["clusters"] if last else None)
        if i >= args.warmup:
            vals.append(last["value"])
            secs.append(time.perf_counter() - t0)
    value = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": "tets/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(secs)),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": workload_config(args, mesh),
            "cpu_baseline": {"value": value, "unit": "tets/s", "cores": 1, "kind": "oracle", "sample": last["sample"],
                             "per_relation_tets_per_s": last["per_relation_tets_per_s"],
                             "extract_s_not_counted": last["extract_s"], "pinned_core": last["pinned_core"]},
            "e2e": {"value": value, "unit": "tets/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def workload_config(args, mesh, extra=None):
    cfg = {"workload": mesh.meta["name"], "config_index": args.config, "dim": mesh.dim,
           "num_vertices": mesh.num_vertices, "num_simplices": mesh.num_simplices,
           "num_clusters": mesh.num_clusters, "batch_clusters": args.batch, "relations": "VT+VV+TT",
           "l2_policy": "inputs+outputs of a step (GBs) far exceed the 126 MB L2; no flush needed"}
    if extra:
        cfg.update(extra)
    return cfg


def library_source_hash() -> str:
    """sha256 (first 16 hex digits) over the CUDA sources of the library and its header, in a fixed order: the key
    that ties an ncu-derived constant in profiles/roofline_traffic.json to the build it was captured from."""
    import hashlib

    csrc = os.path.join(ROOT, "paper_2507_15230_b200", "csrc")
    files = sorted(os.path.join(csrc, f) for f in os.listdir(csrc) if f.endswith((".cu", ".cuh")))
    files.append(os.path.join(ROOT, "include", "gale.h"))
    h = hashlib.sha256()
    for f in files:
        h.update(os.path.basename(f).encode() + b"\0" + open(f, "rb").read() + b"\0")
    return h.hexdigest()[:16]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--n", type=int, default=None, help="grid size override (smaller mesh of the same family)")
    ap.add_argument("--batch", type=int, default=64)
    ap.add_argument("--ring", type=int, default=8, help="device result slots in the device-timed run")
    ap.add_argument("--tile", type=int, default=0)
    ap.add_argument("--streams", type=int, default=1,
                    help="CUDA streams the batches are submitted on in turn (consecutive batches overlap)")
    ap.add_argument("--mask", type=int, default=7, help="relation mask of the device-timed pass (1 VT, 2 VV, 4 TT; 8 VE, 16 VF, 32 EF, "
                    "64 ET, 128 FT build the edge / triangle lists at create); the bench line of record uses 7, other "
                    "values are for per-relation diagnosis (the roofline figures then still count the VT+VV+TT bytes)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "dense", "walk"],
                    help="kernel variant: auto = gale_mesh_create times both on a sample batch and keeps the faster")
    ap.add_argument("--stage-from-t", action="store_true",
                    help="dense kernel: stage T + T_ex and map to local ids in the kernel (A/B of the create-time re-encoding)")
    ap.add_argument("--sustain-s", type=float, default=2.0,
                    help="length of the second, sustained timed region in seconds (0 = skip)")
    ap.add_argument("--consumer", type=int, default=0,
                    help="> 0: also run CriticalPoints (VV + VT) over the whole mesh through the pinned queue with "
                         "this many consumer threads and report the paper's per-stage waiting times (PAPER.md:411)")
    ap.add_argument("--impl", default="gale", choices=["gale", "reference"])
    ap.add_argument("--canonicalize", action="store_true",
                    help="also time gale_canonicalize (SURVEY §8(f)-1) on a device-scrambled copy of the simplices; reported in config")
    ap.add_argument("--boundary", action="store_true",
                    help="also time the boundary look-ups FE / TE / TF over the whole mesh (builds E and F at create); reported in config")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-depth", type=int, default=3, help="pinned queue slots per handle in the e2e leg")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_2507_15230_b200 as gale

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback exists)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    mesh, gen_s = make_workload(args)
    D = mesh.dim + 1
    nC, B = mesh.num_clusters, args.batch
    batches = [np.arange(b, min(nC, b + B), dtype=np.int32) for b in range(0, nC, B)]

    canon = None
    if args.canonicalize:   # the step before the initialization: rows + vertex order scrambled on the device, best of 3
        Tc = torch.from_numpy(mesh.simplices).cuda()
        S = Tc[torch.randperm(Tc.shape[0], device="cuda", generator=torch.Generator(device="cuda").manual_seed(5))].flip(1).contiguous()
        best = float("inf")
        for _ in range(3):
            torch.cuda.synchronize()
            t0 = time.time()
            out, perm = gale.canonicalize(mesh.dim, mesh.num_vertices, S)
            torch.cuda.synchronize()
            best = min(best, time.time() - t0)
        canon = {"canonicalize_s": best, "rows_per_s": mesh.num_simplices / best, "restored": bool(torch.equal(out, Tc))}
        del Tc, S, out, perm
        torch.cuda.empty_cache()

    t0 = time.time()
    gm = gale.GaleMesh(mesh.dim, mesh.num_vertices, mesh.simplices, mesh.cluster_offsets, max_batch_clusters=B,
                       queue_depth=0, device_ring=args.ring, tile_vertices=args.tile,
                       flags={"auto": 0, "dense": gale.KERNEL_DENSE, "walk": gale.KERNEL_WALK}[args.kernel] |
                       (gale.STAGE_FROM_T if args.stage_from_t else 0) |
                       (gale.WITH_EDGES if args.boundary or args.mask & (gale.REL_VE | gale.REL_EF | gale.REL_ET | gale.REL_FT) else 0) |
                       (gale.WITH_FACETS if (args.boundary and mesh.dim == 3) or args.mask & (gale.REL_VF | gale.REL_EF | gale.REL_ET | gale.REL_FT) else 0) |
                       (gale.WITH_COBOUNDARY if args.mask & (gale.REL_EF | gale.REL_ET | gale.REL_FT) else 0))
    create_s = time.time() - t0
    info = gm.info
    bnd = None
    if args.boundary:   # PAPER.md:186-192 look-ups in bulk: one call per relation over every row, CUDA events, best of 3
        bnd = {}
        for name, rel, rows in (("TE", gale.BND_TE, mesh.num_simplices),) + ((("TF", gale.BND_TF, mesh.num_simplices),
                                                                               ("FE", gale.BND_FE, int(info.num_triangles))) if mesh.dim == 3 else ()):
            best = float("inf")
            for _ in range(3):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                out = gm.boundary(rel, 0, rows)
                e1.record()
                torch.cuda.synchronize()
                best = min(best, e0.elapsed_time(e1))
            bnd[name] = {"rows": rows, "ms": best, "entries_per_s": rows * out.shape[1] / (best * 1e-3)}
            del out
        torch.cuda.empty_cache()
    stream = torch.cuda.current_stream()
    # batches are independent (disjoint result slots): submitting them on several streams in turn lets the
    # draining tail of one launch (8,192 blocks = 3.7 waves of resident blocks) overlap the next launch
    sub_streams = [torch.cuda.Stream() for _ in range(args.streams)] if args.streams > 1 else [stream]

    kernel_ms = []

    def one_pass(g, record=False):
        """Submit every batch; pop/release lagging by the ring so the GPU always has work queued."""
        inflight = 0
        for i, ids in enumerate(batches):
            while g.compute(ids, args.mask, stream=sub_streams[i % len(sub_streams)]) == gale.ERR_WOULD_BLOCK:
                st, v = g.pop(-1)
                if record:
                    kernel_ms.append(v.kernel_ms)
                g.release(v)
                inflight -= 1
            inflight += 1
        while inflight:
            st, v = g.pop(-1)
            if record:
                kernel_ms.append(v.kernel_ms)
            g.release(v)
            inflight -= 1

    def fork(ev):
        """the submission streams start after `ev` (recorded on the timing stream)"""
        for ss in sub_streams:
            if ss is not stream:
                ss.wait_event(ev)

    def join():
        """the timing stream waits for everything submitted so far"""
        for ss in sub_streams:
            if ss is not stream:
                done = torch.cuda.Event()
                done.record(ss)
                stream.wait_event(done)

    def barrier():
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        one_pass(gm)
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.1)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    w0 = time.time()
    e0.record(stream)
    fork(e0)
    for _ in range(args.steps):
        one_pass(gm, record=True)
    join()
    e1.record(stream)
    barrier()
    w1 = time.time()
    clocks = sampler.stop(w0, w1)
    ms = e0.elapsed_time(e1)
    ms = max_over_ranks(ms, dist)
    ms_per_step = ms / args.steps
    value = whole_job_value(world, mesh.num_simplices, ms_per_step)

    # second timed region: the same pass repeated for >= --sustain-s seconds (the burst above is 0.1-0.2 s and
    # runs at boost clocks; this one shows what the kernel holds under sustained load, with its own clocks)
    sustained = None
    if args.sustain_s > 0:
        n_sus = max(args.steps, int(np.ceil(args.sustain_s * 1e3 / max(ms_per_step, 1e-3))))
        sampler2 = ClockSampler(local)
        sampler2.start()
        time.sleep(0.1)
        barrier()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        v0 = time.time()
        s0.record(stream)
        fork(s0)
        for _ in range(n_sus):
            one_pass(gm)
        join()
        s1.record(stream)
        barrier()
        v1 = time.time()
        sus_ms = max_over_ranks(s0.elapsed_time(s1), dist) / n_sus
        sustained = {"value": whole_job_value(world, mesh.num_simplices, sus_ms), "unit": "tets/s", "steps": n_sus,
                     "ms_per_step": sus_ms, "timed_region_s": sus_ms * n_sus * 1e-3, "clocks": sampler2.stop(v0, v1)}

    # roofline of the dominant kernel (gale_batch_kernel): algorithmic bytes per launch / avg launch time
    rows = mesh.num_vertices
    alg_bytes = algorithmic_bytes(mesh.dim, mesh.num_simplices, rows, info.vt_nnz, info.vv_nnz, mesh.num_simplices,
                                  len(batches))
    launches = args.steps * len(batches)
    # The library overlaps consecutive launches on two streams, so a launch's own start-to-end event time
    # (kernel_ms) includes the time it shared the GPU with its neighbour. The duration a launch costs is
    # the device-timed region divided by the launches in it; both are reported.
    event_launch_ms = float(np.mean(kernel_ms)) if kernel_ms else None
    avg_launch_ms = ms_per_step / len(batches)
    achieved = alg_bytes / len(batches) / (avg_launch_ms * 1e-3) / 1e9
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        peak, peak_kind = float(json.load(open(peaks_path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    else:
        peak, peak_kind = FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"
    traffic, issue, traffic_note = None, None, None
    build_hash = library_source_hash()
    tpath = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    if os.path.exists(tpath):
        tj = json.load(open(tpath))
        # The ncu constants describe ONE kernel on ONE workload from ONE build: they are emitted only for that launch
        # configuration (walk kernel, config 5, VT + VV + TT, batches of 64, 32-vertex tiles), and the hash of the
        # sources they were captured from travels with them so that a stale constant shows.
        same_launch = (info.kernel_variant == 1 and args.config == 5 and args.mask == 7 and args.n is None and
                       args.batch == 64 and args.tile in (0, 32))
        if same_launch:
            traffic = tj.get("dram_bytes_per_launch")
            traffic_note = {"captured_build_hash": tj.get("build_hash"), "this_build_hash": build_hash,
                            "same_build": tj.get("build_hash") == build_hash}
        # secondary view (the kernel is limited by instruction issue, not by HBM): warp-instructions per
        # launch from the committed ncu capture of this build / the measured launch time, against 4 issue slots per
        # SM per cycle at the SM clock sampled during the timed region
        wi = tj.get("warp_instructions_per_launch")
        if wi and same_launch:
            sms = torch.cuda.get_device_properties(0).multi_processor_count
            mhz = clocks.get("sm_mhz") or clocks.get("sm_max_mhz") or 1965.0
            peak_i = sms * 4 * mhz * 1e6
            issue = {"warp_inst_per_launch": wi, "achieved_ginst_s": wi / (avg_launch_ms * 1e-3) / 1e9,
                     "peak_ginst_s": peak_i / 1e9, "frac": wi / (avg_launch_ms * 1e-3) / peak_i}
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "kernel": ("gale_walk_kernel" if info.kernel_variant == 1 else "gale_batch_kernel") + f"<{D}>", "peak_kind": peak_kind,
                "bytes_per_launch": alg_bytes / len(batches), "avg_launch_ms": avg_launch_ms,
                "avg_launch_ms_is": "CUDA-event time of the timed region / launches in it (2 launches overlap)",
                "event_launch_ms": event_launch_ms,
                "step_gbs": alg_bytes / (ms_per_step * 1e-3) / 1e9,
                "frac_of_8TBs_nominal": achieved / 8000.0, "issue": issue, "traffic_build": traffic_note,
                "build_hash": build_hash}
    gm.destroy()
    del gm

    # end to end through the C ABI with host buffers
    e2e = None
    if not args.no_e2e:
        host_T = torch.from_numpy(mesh.simplices).pin_memory()
        dev_T = torch.empty_like(host_T, device="cuda")
        dev_T.copy_(host_T, non_blocking=True)
        # Two handles over two device copies of the simplex array (double-buffered input): while step i streams
        # its results out of handle i % 2, the input of step i + 1 goes up into the other handle on a copy stream.
        # PCIe is full duplex, so the upload hides behind the result copies; the step is then bound by the D2H link.
        kflag = {"auto": 0, "dense": gale.KERNEL_DENSE, "walk": gale.KERNEL_WALK}[args.kernel] | gale.STREAM_ORDERED
        hs = [gale.GaleMesh(mesh.dim, mesh.num_vertices, dev_T if k == 0 else dev_T.clone(), mesh.cluster_offsets,
                            max_batch_clusters=B, queue_depth=args.e2e_depth, tile_vertices=args.tile, flags=kflag) for k in range(2)]
        d2h = 4 * (2 * (rows + len(batches)) + info.vt_nnz + info.vv_nnz + D * mesh.num_simplices)
        h2d = host_T.numel() * 4
        checksum = 0
        pending = collections.deque()                               # handles in submission order, one entry per batch
        main, up = torch.cuda.current_stream(), torch.cuda.Stream()
        ev_up = [torch.cuda.Event() for _ in hs]
        ev_free = [torch.cuda.Event() for _ in hs]

        def drain_one():
            nonlocal checksum
            g = pending.popleft()
            st, v = g.pop(-1)
            a = g.view_arrays(v)
            checksum += int(a["vt_offsets"][-1]) + int(a["vv_offsets"][-1]) + int(a["tt_indices"][-1])  # host reads
            g.release(v)

        def drain_all():
            while pending:
                drain_one()

        def upload(k):
            """H2D of one step's input from pinned memory into handle k, after the kernels that last read it"""
            up.wait_event(ev_free[k])
            with torch.cuda.stream(up):
                hs[k].simplices.copy_(host_T, non_blocking=True)
                ev_up[k].record(up)

        def submit(k):
            """every batch of one step on handle k; finished batches (of either handle, in submission order) are
            popped, read and released as the bounded queues demand"""
            main.wait_event(ev_up[k])
            for ids in batches:
                while hs[k].compute(ids) == gale.ERR_WOULD_BLOCK:
                    while pending[0] is not hs[k]:
                        drain_one()
                    drain_one()
                pending.append(hs[k])
            ev_free[k].record(main)

        for k in range(2):
            ev_free[k].record(main)
        e2e_steps = max(3, min(args.steps, 6))
        upload(0); submit(0); drain_all()                           # warm-up
        upload(1); submit(1); drain_all()
        barrier()
        t0 = time.perf_counter()
        for i in range(e2e_steps):                                  # every step waits for all of its own results
            upload(i % 2); submit(i % 2); drain_all()
        barrier()
        dt_serial = max_over_ranks((time.perf_counter() - t0) / e2e_steps, dist)
        t0 = time.perf_counter()
        upload(0)
        for i in range(e2e_steps):                                  # steps back to back, next input uploaded meanwhile
            if i + 1 < e2e_steps:
                upload((i + 1) % 2)
            submit(i % 2)
        drain_all()
        barrier()
        dt = max_over_ranks((time.perf_counter() - t0) / e2e_steps, dist)
        e2e = {"value": whole_job_value(world, mesh.num_simplices, dt * 1e3), "unit": "tets/s", "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": dt * 1e3, "steps": e2e_steps,
               "d2h_gbs": d2h / dt / 1e9, "h2d_gbs": h2d / dt / 1e9,
               "serial_value": whole_job_value(world, mesh.num_simplices, dt_serial * 1e3), "serial_ms_per_step": dt_serial * 1e3,
               "what": "every step: H2D of the simplex array from pinned memory, streamed pass (queue_depth=%d)" % args.e2e_depth + ", D2H of every "
                       "CSR batch to pinned slots, pop + read + release on the host. value: steps back to back on two "
                       "handles (double-buffered input: the upload of step i+1 runs on a copy stream under the result "
                       "copies of step i; bound by the D2H link, see d2h_gbs); serial_value: each step uploads, "
                       "computes and drains before the next starts",
               "input_is": "the SAME mesh every step: the handle and its index (the paper's initialization, PAPER.md:178) are "
                           "created once outside the timed region, as the paper's producers are; the batch kernels read that "
                           "index, and of the re-uploaded simplex array only the cross-cluster TT look-ups. The cost of a "
                           "NEW mesh is new_input below",
               "headline": "value (resident index; the paper's setting: initialization once, then relation requests)"}
        for g in hs:
            g.destroy()
        del hs
        torch.cuda.empty_cache()
        # A NEW input every step: upload + initialization (gale_plan_create + gale_mesh_create_planned, workspace
        # allocation included) + the streamed pass with every result copied to the host + destroy.
        def new_input_step():
            nonlocal checksum
            dev_T.copy_(host_T, non_blocking=True)
            t_c = time.perf_counter()
            g = gale.GaleMesh(mesh.dim, mesh.num_vertices, dev_T, mesh.cluster_offsets, max_batch_clusters=B,
                              queue_depth=args.e2e_depth, tile_vertices=args.tile, flags=kflag)
            c_s = time.perf_counter() - t_c
            n_in = 0
            for ids in batches:
                while g.compute(ids) == gale.ERR_WOULD_BLOCK:
                    st, v = g.pop(-1)
                    a = g.view_arrays(v)
                    checksum += int(a["vt_offsets"][-1]) + int(a["vv_offsets"][-1]) + int(a["tt_indices"][-1])
                    g.release(v)
                    n_in -= 1
                n_in += 1
            while n_in:
                st, v = g.pop(-1)
                a = g.view_arrays(v)
                checksum += int(a["vt_offsets"][-1]) + int(a["vv_offsets"][-1]) + int(a["tt_indices"][-1])
                g.release(v)
                n_in -= 1
            g.destroy()
            return c_s

        new_input_step()                                            # warm-up
        barrier()
        t0 = time.perf_counter()
        n_new = 2
        create_warm = [new_input_step() for _ in range(n_new)]
        barrier()
        dt_new = max_over_ranks((time.perf_counter() - t0) / n_new, dist)
        e2e["new_input"] = {"value": whole_job_value(world, mesh.num_simplices, dt_new * 1e3), "unit": "tets/s",
                            "ms_per_step": dt_new * 1e3, "steps": n_new, "create_s_warm": float(np.mean(create_warm)),
                            "what": "every step is a new mesh: H2D of the simplex array, GaleMesh() = initialization on the "
                                    "device + workspace allocation, one streamed pass with every CSR batch copied to pinned "
                                    "host slots and read, destroy"}

    cons = None
    if args.consumer > 0 and rank == 0:
        from paper_2507_15230_b200 import consumer as gc
        mf = mesh if mesh.scalar is not None else meshgen.make_config(args.config, n=args.n, keep_fields=True)
        r = gc.run_critical_points(mf, mf.scalar, consumers=args.consumer, batch=B, queue_depth=4,
                                   kernel_flags={"auto": 0, "dense": gale.KERNEL_DENSE, "walk": gale.KERNEL_WALK}[args.kernel])
        cons = {k: r[k] for k in ("minima", "maxima", "saddles", "regular", "wall_s", "batches", "consumers", "stages_ms", "note", "kernel")}
        cons["what"] = ("CriticalPoints (PAPER.md:292) on the configs' float32 scalar field: VV + VT of every cluster through "
                        "the pinned queue, classified by host consumer threads; stage times are sums over all batches")

    cpu = None
    if rank == 0 and not args.no_cpu_baseline and world == 1:
        o = oracle_sample(mesh)
        cpu = {"value": o["value"], "unit": "tets/s", "cores": 1, "kind": "oracle", "sample": o["sample"],
               "per_relation_tets_per_s": o["per_relation_tets_per_s"], "extract_s_not_counted": o["extract_s"],
               "pinned_core": o["pinned_core"]}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": "tets/s", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "int32", "data": "synthetic",
                "config": workload_config(args, mesh, {"tile_vertices": info.tile_vertices, "num_tiles": info.num_tiles,
                                                       "smem_bytes_per_block": info.smem_bytes,
                                                       "device_ring": args.ring, "parallelism": f"replicas x{world}",
                                                       "mesh_create_s": create_s, "mesh_create_s_is": "first GaleMesh() of the process: CUDA module load, "
                                                       "workspace allocation and the create-time kernel choice included (cold); a warm create is e2e.new_input.create_s_warm",
                                                       "mesh_generate_s": gen_s,
                                                       "kernel": ["dense", "walk"][info.kernel_variant],
                                                       "kernel_choice": args.kernel,
                                                       "create_sample_ms": {"dense": info.tune_dense_ms, "walk": info.tune_walk_ms},
                                                       "block_threads": info.block_threads, "relation_mask": args.mask,
                                                       "index_bytes": info.index_bytes, "workspace_used": info.workspace_used,
                                                       "mesh_bytes": int(mesh.simplices.nbytes),
                                                       **({"canonicalize": canon} if canon else {}),
                                                       **({"boundary": bnd} if bnd else {})}),
                "clocks": clocks, "sustained": sustained, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
                "cpu_baseline": cpu}
        if cons is not None:
            line["consumer"] = cons
        print(json.dumps(line))
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
