"""The scalar-field consumer: Fig. 1's neighbour sum and the critical-point
classification from VV + VT, on the CPU oracle's relations (no GPU), pinned by what the
paper prints, closed forms and a naive re-enumeration; then (gpu) through the pinned queue with consumer
threads and the paper's per-stage waiting-time report."""
import numpy as np
import pytest

import meshgen
import oracle
from paper_2507_15230_b200 import consumer


def _global(m, mask=3):
    g = oracle.relations_global(m.dim, m.num_vertices, m.simplices, mask=mask)
    return {k: (v.astype(np.int32) if k.endswith("_off") else v) for k, v in g.items()}


def test_fig1_neighbour_sum():
    """VV(v0) = [v1, v2, v3]; the derived value of v0 is the sum of their scalars."""
    m = meshgen.toy_two_tets()
    f = np.array([5.0, 1.0, 2.0, 4.0, 8.0], np.float32)
    g = _global(m)
    s = consumer.neighbour_sum(g["vv_off"], g["vv_idx"], f)
    assert s[0] == f[1] + f[2] + f[3]
    assert s[4] == f[1] + f[2] + f[3] and s[1] == f[0] + f[2] + f[3] + f[4]
    assert np.allclose(s, oracle.neighbour_sum(5, g["vv_off"], g["vv_idx"], f))


def test_neighbour_sum_closed_form_and_oracle():
    m = meshgen.make_config(1, keep_fields=True)
    g = _global(m)
    ones = np.ones(m.num_vertices, np.float32)
    deg = consumer.neighbour_sum(g["vv_off"], g["vv_idx"], ones)
    assert deg.max() == 14 and np.array_equal(deg, np.diff(g["vv_off"]))      # interior Kuhn vertex: 14 neighbours
    f = m.scalar.astype(np.float32)
    assert np.allclose(consumer.neighbour_sum(g["vv_off"], g["vv_idx"], f),
                       oracle.neighbour_sum(m.num_vertices, g["vv_off"], g["vv_idx"], f), rtol=1e-6)


_CODE = {oracle.CP_REGULAR: consumer.REGULAR, oracle.CP_MINIMUM: consumer.MINIMUM, oracle.CP_SADDLE: consumer.SADDLE,
         oracle.CP_MAXIMUM: consumer.MAXIMUM}


def _oracle_types(m, f):
    """oracle.critical_points (the plain definition: lower / upper link components by flood fill) as the consumer's codes"""
    return np.array([_CODE[c] for c in oracle.critical_points(m.dim, m.num_vertices, m.simplices, f)], np.uint8)


def test_oracle_critical_points_hand_derived_example():
    """Pin of oracle.critical_points on Fig. 1's mesh (tetrahedra (v0 v1 v2 v3), (v1 v2 v3 v4)) with
    f = (5, 1, 2, 4, 8), derived by hand:
      v0 (5): neighbours v1 v2 v3 all lower, one triangle -> upper link empty                      -> maximum
      v1 (1): neighbours v0 v2 v3 v4 all higher -> lower link empty                                 -> minimum
      v2 (2): lower {v1}; upper {v0, v3, v4}, v0-v3 share the first simplex, v3-v4 the second: 1+1   -> regular
      v3 (4): lower {v1, v2} (adjacent); upper {v0, v4}: v0 and v4 share no simplex: 1 + 2          -> saddle
      v4 (8): neighbours v1 v2 v3 all lower                                                        -> maximum"""
    m = meshgen.toy_two_tets()
    got = oracle.critical_points(3, 5, m.simplices, np.array([5.0, 1.0, 2.0, 4.0, 8.0]))
    assert got == [oracle.CP_MAXIMUM, oracle.CP_MINIMUM, oracle.CP_REGULAR, oracle.CP_SADDLE, oracle.CP_MAXIMUM]
    # ties are broken by vertex id: with a constant field the order is the id order
    flat = oracle.critical_points(3, 5, m.simplices, np.zeros(5))
    assert flat[0] == oracle.CP_MINIMUM and flat[4] == oracle.CP_MAXIMUM and oracle.CP_SADDLE not in flat


@pytest.mark.parametrize("dim,n", [(3, 7), (2, 16)])
def test_oracle_critical_points_linear_function_closed_form(dim, n):
    """Pin of oracle.critical_points: a linear function on a triangulated convex box has exactly one minimum, one
    maximum and no saddle (sub-level sets of a linear function on a convex set are convex, hence connected)."""
    m = meshgen.make_mesh(dim, n, clustering="octree", capacity=200, permute=True, seed=12)
    pos = np.rint(m.coords).astype(np.float64)
    f = pos @ np.array([1.0, np.pi, np.e][:dim])
    got = oracle.critical_points(dim, m.num_vertices, m.simplices, f)
    assert got.count(oracle.CP_MINIMUM) == 1 and got.count(oracle.CP_MAXIMUM) == 1 and got.count(oracle.CP_SADDLE) == 0
    assert got[int(np.argmin(f))] == oracle.CP_MINIMUM and got[int(np.argmax(f))] == oracle.CP_MAXIMUM


@pytest.mark.parametrize("dim,n", [(3, 6), (2, 9)])
def test_critical_points_against_naive_enumeration(dim, n):
    m = meshgen.make_mesh(dim, n, clustering="octree", capacity=60, permute=True, drop_frac=0.15, seed=11)
    g = _global(m)
    f = m.scalar.astype(np.float32)
    got = consumer.critical_points(0, dim + 1, g["vt_off"], g["vt_idx"], g["vv_off"], g["vv_idx"], m.simplices, f)
    assert np.array_equal(got, _oracle_types(m, f))
    assert (got == consumer.SADDLE).any() and (got == consumer.MINIMUM).any()


@pytest.mark.parametrize("dim,n", [(3, 10), (2, 24)])
def test_linear_function_on_a_convex_grid_has_one_minimum_one_maximum_no_saddle(dim, n):
    """A linear function restricted to a triangulated convex box is PL with exactly one minimum, one
    maximum and no saddle (its sub-level sets are convex)."""
    m = meshgen.make_mesh(dim, n, clustering="octree", capacity=200, permute=True, seed=12)
    pos = np.rint(m.coords).astype(np.float64)                      # grid positions (the jitter is +-0.2)
    f = (pos @ np.array([1.0, np.pi, np.e][:dim])).astype(np.float32)
    g = _global(m)
    got = consumer.critical_points(0, dim + 1, g["vt_off"], g["vt_idx"], g["vv_off"], g["vv_idx"], m.simplices, f)
    hist = np.bincount(got, minlength=4)
    assert hist[consumer.MINIMUM] == 1 and hist[consumer.MAXIMUM] == 1 and hist[consumer.SADDLE] == 0
    assert got[np.argmin(f)] == consumer.MINIMUM and got[np.argmax(f)] == consumer.MAXIMUM


def test_run_critical_points_stops_and_raises_when_the_queue_fails(monkeypatch):
    """A fatal pop status (e.g. GALE_ERR_WORKSPACE after a device guard fired) must end the run with the error,
    not leave the producer spinning on back-pressure and the other consumers polling an empty queue (no GPU:
    the handle is a stand-in whose queue fails after the second submitted batch)."""
    import threading

    import paper_2507_15230_b200 as gale

    made = []

    class FailingMesh:
        info = None

        def __init__(self, *a, **k):
            self.lock, self.submitted, self.destroyed = threading.Lock(), 0, False
            made.append(self)

        def compute(self, ids, mask):
            with self.lock:
                if self.submitted >= 2:
                    return gale.ERR_WOULD_BLOCK          # the bounded queue is full and nothing is ever released
                self.submitted += 1
                return gale.OK

        def pop(self, timeout_ms=-1):
            if self.submitted < 2:
                return gale.ERR_EMPTY, None
            raise gale.GaleError(gale.ERR_WORKSPACE, "gale_queue_pop", "device capacity guard fired: code 3")

        def destroy(self):
            self.destroyed = True

    monkeypatch.setattr(gale, "GaleMesh", FailingMesh)
    m = meshgen.make_config(1, keep_fields=True)
    result = {}

    def run():
        try:
            consumer.run_critical_points(m, m.scalar, consumers=3, batch=2)
        except gale.GaleError as e:
            result["error"] = e

    t = threading.Thread(target=run, daemon=True)
    t.start()
    t.join(30)
    assert not t.is_alive()                              # nobody spins forever
    assert result["error"].status == gale.ERR_WORKSPACE and made[0].destroyed


_cfg3_types = []


def _config3_oracle_types():
    """oracle.critical_points of config 3 at n = 32 (about 4 s of python), computed once for both parametrisations"""
    if not _cfg3_types:
        m = meshgen.make_config(3, n=32, keep_fields=True)
        _cfg3_types.append(_oracle_types(m, m.scalar.astype(np.float32)))
    return _cfg3_types[0]


@pytest.mark.gpu
@pytest.mark.parametrize("consumers", [1, 3])
def test_critical_points_through_the_queue(consumers):
    m = meshgen.make_config(3, n=32, keep_fields=True)
    f = m.scalar.astype(np.float32)
    res = consumer.run_critical_points(m, f, consumers=consumers, batch=4, queue_depth=3)
    # the whole path (CUDA relations -> pinned queue -> consumer threads) against the ORACLE's definition of the
    # classification on the oracle's own relations — not against the consumer's classifier fed with oracle relations
    assert np.array_equal(res["types"], _config3_oracle_types())
    assert res["minima"] + res["maxima"] + res["saddles"] + res["regular"] == m.num_vertices
    st = res["stages_ms"]
    assert res["batches"] == (m.num_clusters + 3) // 4
    assert st["kernel_ms"] > 0 and st["d2h_ms"] > 0 and st["consume_ms"] > 0 and st["integrate_ms"] == 0
    assert all(v >= 0 for v in st.values())
