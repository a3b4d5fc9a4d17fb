// gale_consumer.cpp — host-side consumers of the relation queue (the paper's "consumer threads",
// PAPER.md:156 §4.2, :184-198 §4.4): plain C++ that reads the CSR batches gale_queue_pop hands out
// (pinned host memory) together with a per-vertex scalar field. Not part of the GPU hot path; it is what
// the hot path feeds.
//   * neighbour sum: "for each vertex ... a new value is obtained by summing the scalar values of its
//     adjacent vertices" (Fig. 1(c)) — needs VV;
//   * critical points: minima, maxima and saddles of the piecewise-linear scalar field, "requires two
//     vertex-related topological relations, i.e., VV and VT": a vertex is classified by
//     the number of connected components of its lower and upper link (two neighbours are connected when
//     a simplex of the vertex' star contains both); ties of the scalar are broken by the vertex id.
#include <cstdint>
#include <vector>

extern "C" {

// rows [0, n_rows) of a batch: out[r] = sum of scalar[u] over u in VV(row r). offsets are batch-relative.
void gc_neighbour_sum(int64_t n_rows, const int32_t* vv_off, const int32_t* vv_idx, const float* scalar, double* out) {
  for (int64_t r = 0; r < n_rows; ++r) {
    double s = 0.0;
    for (int32_t i = vv_off[r]; i < vv_off[r + 1]; ++i) s += scalar[vv_idx[i]];
    out[r] = s;
  }
}

enum { GC_REGULAR = 0, GC_MINIMUM = 1, GC_MAXIMUM = 2, GC_SADDLE = 3 };

// rows [0, n_rows) are the vertices first_vertex + r. T = the mesh's simplices (D ids each), scalar per
// vertex. out_type[r] in {regular, minimum, maximum, saddle}; counts4 (may be null) accumulates a histogram.
void gc_critical_points(int64_t n_rows, int32_t first_vertex, int D, const int32_t* vt_off, const int32_t* vt_idx,
                        const int32_t* vv_off, const int32_t* vv_idx, const int32_t* T, const float* scalar,
                        uint8_t* out_type, int64_t* counts4) {
  std::vector<int> parent;
  for (int64_t r = 0; r < n_rows; ++r) {
    const int32_t v = first_vertex + int32_t(r);
    const int32_t* nb = vv_idx + vv_off[r];
    const int n = vv_off[r + 1] - vv_off[r];
    parent.resize(size_t(n));
    for (int i = 0; i < n; ++i) parent[size_t(i)] = i;
    auto find = [&](int x) { while (parent[size_t(x)] != x) x = parent[size_t(x)] = parent[size_t(parent[size_t(x)])]; return x; };
    auto lower = [&](int32_t u) { return scalar[u] < scalar[v] || (scalar[u] == scalar[v] && u < v); };
    auto slot = [&](int32_t u) {  // position of u in the sorted neighbour row
      int lo = 0, hi = n;
      while (lo < hi) { const int mid = (lo + hi) >> 1; if (nb[mid] < u) lo = mid + 1; else hi = mid; }
      return lo;
    };
    // neighbours in one simplex of the star are linked when they lie on the same side of v
    for (int32_t i = vt_off[r]; i < vt_off[r + 1]; ++i) {
      const int32_t* s = T + int64_t(vt_idx[i]) * D;
      int first_lo = -1, first_up = -1;
      for (int k = 0; k < D; ++k) {
        if (s[k] == v) continue;
        const int j = slot(s[k]);
        int& anchor = lower(s[k]) ? first_lo : first_up;
        if (anchor < 0) anchor = j; else parent[size_t(find(j))] = find(anchor);
      }
    }
    int comp_lo = 0, comp_up = 0;
    for (int i = 0; i < n; ++i)
      if (find(i) == i) (lower(nb[i]) ? comp_lo : comp_up)++;
    uint8_t t = GC_SADDLE;
    if (comp_lo == 0) t = GC_MINIMUM;        // also isolated vertices
    else if (comp_up == 0) t = GC_MAXIMUM;
    else if (comp_lo == 1 && comp_up == 1) t = GC_REGULAR;
    out_type[r] = t;
    if (counts4) counts4[t]++;
  }
}

}  // extern "C"
