"""Request queues + leader producer with look-ahead.

The paper's consumers do not compute relations themselves: a consumer that needs relation R of a segment
pushes a request into the FIFO queue of R and sleeps on a semaphore; the leader producer pops ALL pending
requests of a queue, adds the segments that follow each requested one ("look-ahead": a
request covers n_b * t_b / t_s consecutive segments), launches one batch, hands the results
over and wakes the consumers. Relations are computed and discarded: the store below is a
small LRU, not a global data structure.

`RelationServer` is that layer over the C ABI: `get(relation, cluster)` blocks until the CSR piece of the
cluster is there. The backend is a function (relation_mask, [cluster ids]) -> list of per-cluster dicts as
`paper_2507_15230_b200.split_batch` returns them; `gale_backend` makes one from a GaleMesh handle (compute +
pop + host copy + release), tests may pass any other."""
from __future__ import annotations

import collections
import threading
import time

import numpy as np

REL_NAMES = {1: "vt", 2: "vv", 4: "tt"}


def gale_backend(gm):
    """Backend over a GaleMesh handle with a pinned queue: one batch per call, results copied out of the
    pinned slot (the only copy: ids are already global, the paper's remap stage does not exist)."""
    import paper_2507_15230_b200 as gale

    def run(mask, ids):
        host = gm.run_batch(ids, mask)
        return gale.split_batch(host, gm.D), dict(kernel_ms=host["kernel_ms"], d2h_ms=host["d2h_ms"], prep_ms=host["prep_ms"])
    return run


class RelationServer:
    def __init__(self, backend, num_clusters: int, *, max_batch: int = 64, lookahead: int = 4, store_clusters: int = 512):
        self.backend, self.nC = backend, int(num_clusters)
        self.max_batch, self.lookahead = int(max_batch), max(1, int(lookahead))
        self.queues = {r: collections.deque() for r in REL_NAMES}          # one FIFO per relation
        self.store = {r: collections.OrderedDict() for r in REL_NAMES}     # cluster -> result, LRU, bounded
        self.store_cap = int(store_clusters)
        self.cv = threading.Condition()
        self.stop = False
        self.error = None                                                  # the exception that ended the leader, if any
        self.stats = dict(requests=0, hits=0, launches=0, clusters_computed=0, lookahead_used=0,
                          queue_lengths=[], enqueue_ms=0.0, in_queue_ms=0.0, prep_ms=0.0, kernel_ms=0.0, d2h_ms=0.0,
                          integrate_ms=0.0)
        self._lookahead_pending = {r: set() for r in REL_NAMES}
        self.leader = threading.Thread(target=self._lead, daemon=True)
        self.leader.start()

    # ---- consumer side ---------------------------------------------------------------------------------
    def get(self, relation: int, cluster: int):
        """Relation `relation` (1 VT, 2 VV, 4 TT) of `cluster`: (offsets, indices) for VT / VV, [rows, D] for TT."""
        assert relation in REL_NAMES and 0 <= cluster < self.nC
        t0 = time.perf_counter()
        with self.cv:
            self.stats["requests"] += 1
            hit = self.store[relation].get(cluster)
            if hit is not None:
                self.store[relation].move_to_end(cluster)
                self.stats["hits"] += 1
                if cluster in self._lookahead_pending[relation]:
                    self._lookahead_pending[relation].discard(cluster)
                    self.stats["lookahead_used"] += 1
                return hit
            req = dict(cluster=cluster, t_push=time.perf_counter(), result=None)
            self.queues[relation].append(req)                               # push under the lock
            self.stats["enqueue_ms"] += 1e3 * (time.perf_counter() - t0)
            self.cv.notify_all()
            while req["result"] is None and req.get("error") is None and not self.stop:   # the semaphore of the paper
                self.cv.wait(0.05)
            if req["result"] is None:
                err = req.get("error") or self.error
                if err is not None:                                         # the leader producer failed: every waiter learns why
                    raise RuntimeError(f"RelationServer: the leader producer failed: {err!r}") from err
                raise RuntimeError("RelationServer stopped")
            return req["result"]

    # ---- leader producer -------------------------------------------------------------------------------
    def _lead(self):
        """Leader thread: serves until close(). A failing backend (a GaleError from compute / pop, anything else) must
        not leave consumers asleep: the exception is handed to every pending request, the server stops, and get()
        re-raises it in the consumers' threads."""
        work = {}
        try:
            self._serve(work)
        except BaseException as e:   # noqa: BLE001 - handed over to the consumers, not swallowed
            with self.cv:
                self.error = e
                self.stop = True
                for reqs in work.values():
                    for rq in reqs:
                        if rq["result"] is None:
                            rq["error"] = e
                for q in self.queues.values():
                    for rq in q:
                        rq["error"] = e
                    q.clear()
                self.cv.notify_all()

    def _serve(self, work):
        while True:
            work.clear()
            with self.cv:
                while not self.stop and not any(self.queues.values()):
                    self.cv.wait(0.05)
                if self.stop:
                    return
                for r, q in self.queues.items():                            # pop ALL pending requests
                    if q:
                        self.stats["queue_lengths"].append(len(q))
                        work[r] = list(q)
                        q.clear()
            for r, reqs in work.items():
                now = time.perf_counter()
                want, asked = [], set()
                for rq in reqs:
                    asked.add(rq["cluster"])
                    for c in range(rq["cluster"], min(self.nC, rq["cluster"] + self.lookahead)):   # look-ahead
                        if c not in want and c not in self.store[r]:
                            want.append(c)
                results = {}
                for b in range(0, len(want), self.max_batch):
                    ids = want[b:b + self.max_batch]
                    pieces, tm = self.backend(r, ids)
                    t_int = time.perf_counter()
                    for c, piece in zip(ids, pieces):
                        results[c] = piece[REL_NAMES[r]]
                    with self.cv:
                        self.stats["launches"] += 1
                        self.stats["clusters_computed"] += len(ids)
                        for k in ("prep_ms", "kernel_ms", "d2h_ms"):
                            self.stats[k] += float(tm.get(k, 0.0))
                        self.stats["integrate_ms"] += 1e3 * (time.perf_counter() - t_int)
                with self.cv:
                    for c, res in results.items():
                        self.store[r][c] = res
                        if c not in asked:
                            self._lookahead_pending[r].add(c)
                    # hand the results over BEFORE discarding: a requested cluster that an earlier look-ahead had
                    # already cached is not in `results`, and a small store may evict it in this very pass
                    for rq in reqs:
                        c = rq["cluster"]
                        res = results.get(c)
                        if res is None:
                            res = self.store[r].get(c)
                        if res is None:
                            raise RuntimeError(f"no result for relation {r} of cluster {c}")
                        rq["result"] = res
                        self.stats["in_queue_ms"] += 1e3 * (now - rq["t_push"])
                    while len(self.store[r]) > self.store_cap:               # compute and discard
                        old, _ = self.store[r].popitem(last=False)
                        self._lookahead_pending[r].discard(old)
                    self.cv.notify_all()

    def close(self):
        with self.cv:
            self.stop = True
            self.cv.notify_all()
        self.leader.join(timeout=5)

    def summary(self) -> dict:
        s = dict(self.stats)
        ql = s.pop("queue_lengths")
        s["queue_length_mean"] = float(np.mean(ql)) if ql else 0.0
        s["queue_length_median"] = float(np.median(ql)) if ql else 0.0
        s["hit_rate"] = s["hits"] / max(1, s["requests"])
        return s
