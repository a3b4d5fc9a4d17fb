"""Request queues + leader producer with look-ahead: the host
logic on the CPU with the oracle as backend (no GPU), then (gpu) over the C ABI with several consumer threads."""
import threading

import numpy as np
import pytest

import meshgen
import oracle
from paper_2507_15230_b200.consumer.requests import RelationServer, gale_backend


def _oracle_backend(m, log):
    def run(mask, ids):
        log.append((mask, list(ids)))
        return oracle.cluster_results(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, ids, mask=mask), {}
    return run


def _same(a, b):
    if isinstance(a, tuple):
        return np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    return np.array_equal(a, b)


def test_lookahead_batches_and_discards():
    m = meshgen.make_config(3, n=24)                     # several clusters
    nC = m.num_clusters
    assert nC >= 8
    log = []
    srv = RelationServer(_oracle_backend(m, log), nC, max_batch=64, lookahead=4, store_clusters=6)
    ref = oracle.cluster_results(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, range(nC))
    for c in range(8):                                   # a consumer sweeping the clusters in order
        assert _same(srv.get(2, c), ref[c]["vv"])
    s = srv.summary()
    assert [ids for (mask, ids) in log if mask == 2] == [[0, 1, 2, 3], [4, 5, 6, 7]]   # one launch per 4 requests
    assert s["requests"] == 8 and s["hits"] == 6 and s["lookahead_used"] == 6 and s["launches"] == 2
    assert _same(srv.get(4, 5), ref[5]["tt"])            # another relation has its own queue and store
    assert log[-1] == (4, [5, 6, 7, 8][:min(4, nC - 5)])
    assert len(srv.store[2]) <= 6                        # compute and discard: the store is bounded
    srv.get(2, 0)                                        # evicted by now: computed again
    assert log[-1][0] == 2 and log[-1][1][0] == 0
    srv.close()


def test_leader_pops_all_pending_requests():
    m = meshgen.make_config(3, n=24)
    nC = m.num_clusters
    log, gate = [], threading.Event()

    def slow_backend(mask, ids):
        gate.wait(5)                                     # hold the leader so that requests pile up in the queue
        return _oracle_backend(m, log)(mask, ids)

    srv = RelationServer(slow_backend, nC, lookahead=1)
    ref = oracle.cluster_results(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, range(nC), mask=1)
    out = {}

    def consumer(c):
        out[c] = srv.get(1, c)

    first = threading.Thread(target=consumer, args=(0,))
    first.start()
    import time
    time.sleep(0.2)                                      # the leader is now inside the backend with request 0
    rest = [threading.Thread(target=consumer, args=(c,)) for c in (3, 5, 6)]
    for t in rest:
        t.start()
    time.sleep(0.2)
    gate.set()
    for t in [first] + rest:
        t.join(10)
    assert [ids for _, ids in log] == [[0], [3, 5, 6]]   # the three pending requests went out as ONE batch
    for c in (0, 3, 5, 6):
        assert _same(out[c], ref[c]["vt"])
    assert srv.summary()["queue_length_mean"] == 2.0     # queue lengths seen by the leader: 1 and 3
    srv.close()


def test_failing_backend_wakes_every_consumer_with_the_error():
    """A backend error (e.g. a GaleError from compute / pop) ends the leader; nobody may stay asleep in get()."""
    import time

    class Boom(RuntimeError):
        pass

    def backend(mask, ids):
        time.sleep(0.2)                                  # let more requests pile up behind the one being served
        raise Boom("device guard fired")

    srv = RelationServer(backend, 16, lookahead=2)
    errors = {}

    def consumer(c):
        try:
            srv.get(1, c)
        except RuntimeError as e:
            errors[c] = e

    ts = [threading.Thread(target=consumer, args=(c,), daemon=True) for c in (0, 5, 9)]
    ts[0].start()
    time.sleep(0.05)
    for t in ts[1:]:
        t.start()
    for t in ts:
        t.join(10)
        assert not t.is_alive()                          # the served request AND the queued ones woke up
    assert sorted(errors) == [0, 5, 9]
    for e in errors.values():
        assert isinstance(e.__cause__, Boom) and "device guard fired" in str(e)
    with pytest.raises(RuntimeError, match="device guard fired"):   # later requests fail at once, too
        srv.get(2, 1)
    srv.close()


def test_store_smaller_than_the_lookahead_window():
    """store_clusters < lookahead x consumers: a request whose cluster an earlier look-ahead cached while it waited
    in the queue is served from the store — and must be served before that pass evicts the cluster again."""
    import time

    m = meshgen.make_config(3, n=24)
    nC = m.num_clusters
    assert nC >= 6
    log, gate = [], threading.Event()

    def slow_backend(mask, ids):
        gate.wait(5)
        return _oracle_backend(m, log)(mask, ids)

    srv = RelationServer(slow_backend, nC, lookahead=2, store_clusters=1)
    ref = oracle.cluster_results(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, range(nC), mask=1)
    out = {}

    def consumer(c):
        out[c] = srv.get(1, c)

    first = threading.Thread(target=consumer, args=(0,), daemon=True)
    first.start()
    time.sleep(0.2)                                      # the leader is computing clusters 0, 1 for request 0
    rest = [threading.Thread(target=consumer, args=(c,), daemon=True) for c in (1, 4)]   # 1 is not in the store yet: queued
    for t in rest:
        t.start()
    time.sleep(0.2)
    gate.set()
    for t in [first] + rest:
        t.join(10)
        assert not t.is_alive()
    # second pass: 1 was cached by the first (the store keeps {1}), so only its look-ahead and 4's window are
    # computed; storing those three evicts 1 in the same pass
    assert [ids for _, ids in log] == [[0, 1], [2, 4, 5]]
    assert 1 not in srv.store[1] and len(srv.store[1]) == 1
    for c in (0, 1, 4):
        assert _same(out[c], ref[c]["vt"])
    srv.close()


@pytest.mark.gpu
def test_request_queues_over_the_c_abi():
    import paper_2507_15230_b200 as gale

    m = meshgen.make_config(3, n=32)
    gm = gale.GaleMesh(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, max_batch_clusters=16, queue_depth=2)
    srv = RelationServer(gale_backend(gm), m.num_clusters, max_batch=16, lookahead=4)
    ref = oracle.cluster_results(m.dim, m.num_vertices, m.simplices, m.cluster_offsets, range(m.num_clusters))
    bad = []

    def consumer(k):
        rng = np.random.default_rng(k)
        start = int(rng.integers(0, m.num_clusters))
        for i in range(12):
            c = (start + i) % m.num_clusters
            for rel, key in ((2, "vv"), (1, "vt"), (4, "tt")):
                if not _same(srv.get(rel, c), ref[c][key]):
                    bad.append((k, rel, c))

    th = [threading.Thread(target=consumer, args=(k,)) for k in range(4)]
    for t in th:
        t.start()
    for t in th:
        t.join(60)
    s = srv.summary()
    srv.close()
    gm.destroy()
    assert not bad
    assert s["requests"] == 4 * 12 * 3 and s["hit_rate"] > 0.3 and s["kernel_ms"] > 0 and s["launches"] < s["requests"]
