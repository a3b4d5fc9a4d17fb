// gale_oracle — CPU oracle for the GALE relation hot path. TEST INFRASTRUCTURE ONLY.
//
// Plain, single-threaded, obviously-correct C++ restatement of the relation *definitions*
// (§2.2 "Topological Relations"; §4.6 "no duplicates"; §4.3
// internal/external rule; readings of SURVEY.md §8(c), listed in DESIGN.md §Readings).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
// call this. It shares no code, header, table or helper with the CUDA path
// (paper_2507_15230_b200/csrc) and neither includes the other.
//
// Parity pins (tests/test_oracle_pins.py, all `-m "not gpu"`): Fig. 4's stated facts for I_T / T_ex /
// the edge intervals (tests/golden/fig4_mesh.txt), Fig. 1 toy (PAPER.md:60-64,
// tests/golden/fig1_toy.txt), brute-force enumeration below (go_brute_*), scipy.sparse transposes /
// products, Kuhn-grid closed forms, Euler characteristic, TT symmetry, clustering independence.
// Nothing here is "parity unpinned".
//
// Input contract ("canonical mesh"): D = dim+1 vertices per simplex, rows of T
// strictly ascending (C1), rows strictly ascending lexicographically (C2), ids in [0,nV) (C3),
// every facet has at most two cofaces (C4). Cluster c owns vertices [o[c], o[c+1]) (PAPER.md:178,
// Alg. 1 line 3 PAPER.md:243) and the *internal* simplices {t : o[c] <= T[t][0] < o[c+1]}
// ("internal ... iff the vertex with the lowest index also belongs to S_i").
//
// Definitions (global; ids are global; every row ascending):
//   VT(v)    = all t with v in T[t]                                    (coboundary)
//   VV(v)    = all u != v sharing some simplex with v, no duplicates   (Alg. 1 :239-249)
//   TT(t)[k] = the t' != t whose vertex set contains T[t] \ {T[t][k]}, else -1  (adjacency, :49)
#include <algorithm>
#include <array>
#include <chrono>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

struct Relations {
  int D = 0;
  int64_t nV = 0, nT = 0;
  std::vector<int64_t> vt_off, vv_off;   // [nV+1]
  std::vector<int32_t> vt_idx, vv_idx;
  std::vector<int32_t> tt;               // [nT*D]
  std::vector<int64_t> first_tet;        // [nV+1]: first t with T[t][0] >= v   (I_T)
  int status = 0;
  double seconds[3] = {0, 0, 0};         // wall time of compute_vt / compute_vv / compute_tt (reporting only)
};

enum { GO_OK = 0, GO_NOT_CANONICAL = -2, GO_NONMANIFOLD = -4 };

int check_canonical(int D, int64_t nV, int64_t nT, const int32_t* T) {
  for (int64_t t = 0; t < nT; ++t) {
    const int32_t* r = T + t * D;
    if (r[0] < 0 || r[D - 1] >= nV) return GO_NOT_CANONICAL;
    for (int k = 1; k < D; ++k)
      if (r[k] <= r[k - 1]) return GO_NOT_CANONICAL;
    if (t > 0 && !std::lexicographical_compare(r - D, r, r, r + D)) return GO_NOT_CANONICAL;
  }
  return GO_OK;
}

// VT: "for t ascending, for k: VT[T[t][k]].push_back(t)"
void compute_vt(Relations& R, const int32_t* T) {
  const int D = R.D;
  R.vt_off.assign(R.nV + 1, 0);
  for (int64_t i = 0; i < R.nT * D; ++i) ++R.vt_off[T[i] + 1];
  for (int64_t v = 0; v < R.nV; ++v) R.vt_off[v + 1] += R.vt_off[v];
  R.vt_idx.resize(R.nT * D);
  std::vector<int64_t> cur(R.vt_off.begin(), R.vt_off.end() - 1);
  for (int64_t t = 0; t < R.nT; ++t)
    for (int k = 0; k < D; ++k) R.vt_idx[cur[T[t * D + k]]++] = int32_t(t);
}

// VV: push every ordered pair (v,u), u != v, of every simplex; per row sort + unique.
void compute_vv(Relations& R, const int32_t* T) {
  const int D = R.D;
  std::vector<int64_t> off(R.nV + 1, 0);
  for (int64_t i = 0; i < R.nT * D; ++i) off[T[i] + 1] += D - 1;
  for (int64_t v = 0; v < R.nV; ++v) off[v + 1] += off[v];
  std::vector<int32_t> all(off[R.nV]);
  std::vector<int64_t> cur(off.begin(), off.end() - 1);
  for (int64_t t = 0; t < R.nT; ++t)
    for (int k = 0; k < D; ++k)
      for (int j = 0; j < D; ++j)
        if (j != k) all[cur[T[t * D + k]]++] = T[t * D + j];
  R.vv_off.assign(R.nV + 1, 0);
  R.vv_idx.clear();
  for (int64_t v = 0; v < R.nV; ++v) {
    int32_t* b = all.data() + off[v];
    int32_t* e = all.data() + off[v + 1];
    std::sort(b, e);
    e = std::unique(b, e);
    R.vv_idx.insert(R.vv_idx.end(), b, e);
    R.vv_off[v + 1] = int64_t(R.vv_idx.size());
  }
}

// TT: list every facet (T[t] minus its k-th vertex) with (t,k); sort by facet; a facet listed
// twice joins its two cofaces, once = boundary (-1), more = not a manifold (C4).
template <int D>
int compute_tt(Relations& R, const int32_t* T) {
  struct Rec {
    std::array<int32_t, D - 1> f;
    int32_t t, k;
  };
  std::vector<Rec> rec(R.nT * D);
  for (int64_t t = 0; t < R.nT; ++t)
    for (int k = 0; k < D; ++k) {
      Rec& r = rec[t * D + k];
      int o = 0;
      for (int j = 0; j < D; ++j)
        if (j != k) r.f[o++] = T[t * D + j];
      r.t = int32_t(t);
      r.k = k;
    }
  std::sort(rec.begin(), rec.end(), [](const Rec& a, const Rec& b) { return a.f != b.f ? a.f < b.f : a.t < b.t; });
  R.tt.assign(R.nT * D, -1);
  for (size_t i = 0; i < rec.size();) {
    size_t j = i + 1;
    while (j < rec.size() && rec[j].f == rec[i].f) ++j;
    if (j - i > 2) return GO_NONMANIFOLD;
    if (j - i == 2) {
      R.tt[int64_t(rec[i].t) * D + rec[i].k] = rec[i + 1].t;
      R.tt[int64_t(rec[i + 1].t) * D + rec[i + 1].k] = rec[i].t;
    }
    i = j;
  }
  return GO_OK;
}

void compute_first_tet(Relations& R, const int32_t* T) {
  R.first_tet.assign(R.nV + 1, 0);
  for (int64_t t = 0; t < R.nT; ++t) ++R.first_tet[T[t * R.D] + 1];
  for (int64_t v = 0; v < R.nV; ++v) R.first_tet[v + 1] += R.first_tet[v];
}

Relations* compute_all(int D, int64_t nV, int64_t nT, const int32_t* T, uint32_t mask) {
  Relations* R = new Relations;
  R->D = D;
  R->nV = nV;
  R->nT = nT;
  R->status = check_canonical(D, nV, nT, T);
  if (R->status != GO_OK) return R;
  compute_first_tet(*R, T);
  using clk = std::chrono::steady_clock;
  auto secs = [](clk::time_point a, clk::time_point b) { return std::chrono::duration<double>(b - a).count(); };
  clk::time_point t0 = clk::now();
  if (mask & 1) compute_vt(*R, T);
  clk::time_point t1 = clk::now();
  if (mask & 2) compute_vv(*R, T);
  clk::time_point t2 = clk::now();
  if (mask & 4) R->status = D == 4 ? compute_tt<4>(*R, T) : compute_tt<3>(*R, T);
  clk::time_point t3 = clk::now();
  R->seconds[0] = secs(t0, t1); R->seconds[1] = secs(t1, t2); R->seconds[2] = secs(t2, t3);  // timers only: no arithmetic
  return R;
}

}  // namespace

extern "C" {

// ---- global relations ---------------------------------------------------------------------------
// mask: 1 = VT, 2 = VV, 4 = TT. Returns an owned handle (free with go_free); go_status() != 0 means
// the input broke the contract (-2 not canonical, -4 non-manifold facet).
void* go_compute_global(int dim, int64_t nV, int64_t nT, const int32_t* T, uint32_t mask) {
  return compute_all(dim + 1, nV, nT, T, mask);
}
int go_status(void* h) { return static_cast<Relations*>(h)->status; }
void go_free(void* h) { delete static_cast<Relations*>(h); }
const int64_t* go_vt_offsets(void* h) { return static_cast<Relations*>(h)->vt_off.data(); }
const int32_t* go_vt_indices(void* h) { return static_cast<Relations*>(h)->vt_idx.data(); }
const int64_t* go_vv_offsets(void* h) { return static_cast<Relations*>(h)->vv_off.data(); }
const int32_t* go_vv_indices(void* h) { return static_cast<Relations*>(h)->vv_idx.data(); }
const int32_t* go_tt(void* h) { return static_cast<Relations*>(h)->tt.data(); }
const int64_t* go_first_tet(void* h) { return static_cast<Relations*>(h)->first_tet.data(); }
int64_t go_vv_nnz(void* h) { return int64_t(static_cast<Relations*>(h)->vv_idx.size()); }
// Wall time the three relation routines took inside go_compute_* (for bench.py's cpu_baseline split).
void go_seconds(void* h, double* out3) {
  for (int i = 0; i < 3; ++i) out3[i] = static_cast<Relations*>(h)->seconds[i];
}

// ---- restriction to a set of clusters (for meshes too large for the global pass) -----------------
// Exactness: let W = vertices of the selected clusters plus every vertex of their internal
// simplices. A simplex incident to a selected vertex has a vertex in W; a simplex sharing a facet
// with an internal simplex t has D-1 >= 1 vertices of t, all in W. So the definitions evaluated on
// the sub-mesh {t : T[t] meets W} give exactly the global VT/VV rows of the selected vertices and
// the global TT rows of the selected internal simplices. The sub-mesh keeps ascending global order,
// so sorted rows stay sorted after mapping sub-mesh ids back (gid).
// Outputs: handle over the sub-mesh + gid array (go_sub_gid). Rows outside the selection are
// *not* meaningful and must not be read.
struct SubMesh {
  Relations* R = nullptr;
  std::vector<int32_t> gid;  // sub-mesh simplex -> global simplex id
  std::vector<int32_t> Tsub;
  double extract_seconds = 0;  // the two whole-mesh scans that build the sub-mesh (reporting only)
};

void* go_compute_restricted(int dim, int64_t nV, int64_t nT, const int32_t* T, int32_t nC,
                            const int32_t* offsets, int32_t nSel, const int32_t* sel, uint32_t mask) {
  const int D = dim + 1;
  (void)nC;
  const auto t_begin = std::chrono::steady_clock::now();
  std::vector<uint8_t> inW(nV, 0);
  for (int32_t i = 0; i < nSel; ++i)
    for (int32_t v = offsets[sel[i]]; v < offsets[sel[i] + 1]; ++v) inW[v] = 1;
  std::vector<uint8_t> inSel(inW);
  for (int64_t t = 0; t < nT; ++t)
    if (inSel[T[t * D]])
      for (int k = 1; k < D; ++k) inW[T[t * D + k]] = 1;
  SubMesh* S = new SubMesh;
  for (int64_t t = 0; t < nT; ++t) {
    bool hit = false;
    for (int k = 0; k < D; ++k) hit |= inW[T[t * D + k]] != 0;
    if (hit) {
      S->gid.push_back(int32_t(t));
      S->Tsub.insert(S->Tsub.end(), T + t * D, T + t * D + D);
    }
  }
  S->extract_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
  S->R = compute_all(D, nV, int64_t(S->gid.size()), S->Tsub.data(), mask);
  return S;
}
void* go_sub_relations(void* s) { return static_cast<SubMesh*>(s)->R; }
const int32_t* go_sub_gid(void* s) { return static_cast<SubMesh*>(s)->gid.data(); }
int64_t go_sub_size(void* s) { return int64_t(static_cast<SubMesh*>(s)->gid.size()); }
double go_sub_extract_seconds(void* s) { return static_cast<SubMesh*>(s)->extract_seconds; }
void go_sub_free(void* s) {
  SubMesh* S = static_cast<SubMesh*>(s);
  delete S->R;
  delete S;
}

// ---- per-cluster slice (SURVEY.md §8(c) "Per-cluster result") --------------------------------------
// Rows v = lo..hi-1 of a vertex relation as CSR starting at 0. map (may be null) renames the
// stored simplex ids (sub-mesh -> global). Returns nnz. off_out has hi-lo+1 entries.
int64_t go_slice_rows(const int64_t* off, const int32_t* idx, int64_t lo, int64_t hi, const int32_t* map,
                      int32_t* off_out, int32_t* idx_out) {
  const int64_t base = off[lo];
  for (int64_t v = lo; v <= hi; ++v) off_out[v - lo] = int32_t(off[v] - base);
  const int64_t nnz = off[hi] - base;
  if (idx_out)
    for (int64_t i = 0; i < nnz; ++i) idx_out[i] = map ? map[idx[base + i]] : idx[base + i];
  return nnz;
}
// TT rows of simplices [t_lo, t_hi) (ids of the handle's own mesh); entries renamed through map.
void go_slice_tt(const int32_t* tt, int D, int64_t t_lo, int64_t t_hi, const int32_t* map, int32_t* out) {
  for (int64_t i = t_lo * D; i < t_hi * D; ++i) out[i - t_lo * D] = (tt[i] < 0 || !map) ? tt[i] : map[tt[i]];
}

// ---- initialization data of a segment -----------------------------------------
// Plain scans over all simplices; a segment is the vertex range [lo, hi).
// I_T: the internal simplices of the segment, {t : lo <= T[t][0] < hi} ("internal ... iff the vertex with
// the lowest index also belongs to S_i", :172), are a contiguous id range by C2; out2 = {first, last+1}
// (first = last+1 = number of simplices with a lower lowest vertex when there is none).
void go_internal_range(int dim, int64_t nT, const int32_t* T, int64_t lo, int64_t hi, int64_t* out2) {
  const int D = dim + 1;
  int64_t below = 0, inside = 0;
  for (int64_t t = 0; t < nT; ++t) {
    if (T[t * D] < lo) ++below;
    else if (T[t * D] < hi) ++inside;
  }
  out2[0] = below;
  out2[1] = below + inside;
}
// T_ex: the external simplices of the segment, ascending: simplices with a vertex in [lo, hi) whose
// lowest vertex is not in it ("external to all other intersecting segments", :172; "T_ex encodes the list
// of external tetrahedra for each segment", :178). out may be null (count only). Returns the count.
int64_t go_external_list(int dim, int64_t nT, const int32_t* T, int64_t lo, int64_t hi, int32_t* out) {
  const int D = dim + 1;
  int64_t n = 0;
  for (int64_t t = 0; t < nT; ++t) {
    const int32_t* r = T + t * D;
    if (r[0] >= lo && r[0] < hi) continue;  // internal
    bool touches = false;
    for (int k = 1; k < D; ++k) touches |= (r[k] >= lo && r[k] < hi);
    if (touches) {
      if (out) out[n] = int32_t(t);
      ++n;
    }
  }
  return n;
}

// ---- edges, triangles and the coboundary relations VE / VF (Table 1 :53-58) ----------
// E = every unique combination of two vertices of a simplex, F = of three ("all unique combinations of two
// vertices (edges) and three vertices (triangles) are stored in sorted indexed lists (E and F) based on
// vertex indices", :178). Reading: each combination ascending, the list in ascending
// lexicographic order, the id of an edge / triangle = its position. A sub-simplex is internal to the
// segment of its lowest vertex (:172), so the interval arrays are I_E[v] / I_F[v] = number of edges /
// triangles whose lowest vertex is below v. For a 2-D mesh F = T.
}  // extern "C" (templates below)
struct SubSimplices {
  int K = 0;                      // vertices per sub-simplex: 2 (edges) or 3 (triangles)
  std::vector<int32_t> list;      // [n*K]
  std::vector<int64_t> first;     // [nV+1] interval array per vertex
  std::vector<int64_t> v_off;     // [nV+1] VE / VF offsets
  std::vector<int32_t> v_idx;     // VE / VF indices (ids of the sub-simplices containing v, ascending)
};
template <int K>
static SubSimplices* enumerate_sub(int D, int64_t nV, int64_t nT, const int32_t* T) {
  using Key = std::array<int32_t, K>;
  std::vector<Key> all;
  for (int64_t t = 0; t < nT; ++t) {
    const int32_t* r = T + t * D;
    if (K == 2) {
      for (int i = 0; i < D; ++i)
        for (int j = i + 1; j < D; ++j) { Key k{}; k[0] = r[i]; k[1] = r[j]; all.push_back(k); }
    } else {
      for (int i = 0; i < D; ++i)
        for (int j = i + 1; j < D; ++j)
          for (int l = j + 1; l < D; ++l) { Key k{}; k[0] = r[i]; k[1] = r[j]; k[2] = r[l]; all.push_back(k); }
    }
  }
  std::sort(all.begin(), all.end());
  all.erase(std::unique(all.begin(), all.end()), all.end());
  SubSimplices* S = new SubSimplices;
  S->K = K;
  S->list.resize(all.size() * K);
  S->first.assign(nV + 1, 0);
  std::vector<int64_t> deg(nV + 1, 0);
  for (size_t i = 0; i < all.size(); ++i) {
    for (int k = 0; k < K; ++k) { S->list[i * K + k] = all[i][k]; ++deg[all[i][k] + 1]; }
    ++S->first[all[i][0] + 1];
  }
  for (int64_t v = 0; v < nV; ++v) { S->first[v + 1] += S->first[v]; deg[v + 1] += deg[v]; }
  S->v_off = deg;
  S->v_idx.resize(all.size() * K);
  std::vector<int64_t> cur(deg.begin(), deg.end() - 1);
  for (size_t i = 0; i < all.size(); ++i)          // ids ascending => every row ascending
    for (int k = 0; k < K; ++k) S->v_idx[cur[all[i][k]]++] = int32_t(i);
  return S;
}
extern "C" {
void* go_enumerate_sub(int dim, int K, int64_t nV, int64_t nT, const int32_t* T) {
  if (K == 2) return enumerate_sub<2>(dim + 1, nV, nT, T);
  if (K == 3) return enumerate_sub<3>(dim + 1, nV, nT, T);
  return nullptr;
}
int64_t go_sub_count(void* h) { SubSimplices* S = static_cast<SubSimplices*>(h); return int64_t(S->list.size()) / S->K; }
const int32_t* go_sub_list(void* h) { return static_cast<SubSimplices*>(h)->list.data(); }
const int64_t* go_sub_first(void* h) { return static_cast<SubSimplices*>(h)->first.data(); }
const int64_t* go_sub_v_off(void* h) { return static_cast<SubSimplices*>(h)->v_off.data(); }
const int32_t* go_sub_v_idx(void* h) { return static_cast<SubSimplices*>(h)->v_idx.data(); }
void go_sub_release(void* h) { delete static_cast<SubSimplices*>(h); }

// Coboundary relations between sub-simplices ("the coboundary relation R_{k,p}, k < p, maps a
// k-simplex to the p-simplices incident in it"; Table 1 :53-58): rows = the sorted list of (from)-vertex
// sub-simplices (from = 2 edges, 3 triangles), entries = ascending ids of the (to)-vertex simplices that
// contain them (to = 3: triangles of the sorted list F; to = D: the simplices of T). EF = (2,3), ET = (2,D),
// FT = (3,D). Plain: for every containing simplex in ascending id order, look each of its sub-simplices up
// in the sorted row list and append the id.
}  // extern "C" (templates below)
struct Cobound {
  std::vector<int64_t> off;
  std::vector<int32_t> idx;
};
template <int KF>
static void cobound_fill(Cobound& C, const std::vector<int32_t>& rows, int KT, int64_t nCols, const int32_t* cols) {
  using Key = std::array<int32_t, KF>;
  const int64_t nRows = int64_t(rows.size()) / KF;
  auto row_id = [&](const Key& k) {
    int64_t lo = 0, hi = nRows;
    while (lo < hi) {
      const int64_t mid = (lo + hi) / 2;
      Key r;
      for (int i = 0; i < KF; ++i) r[i] = rows[mid * KF + i];
      if (r < k) lo = mid + 1; else hi = mid;
    }
    return lo;
  };
  std::vector<std::vector<int32_t>> lists(nRows);
  std::vector<int> pick(KF);
  for (int64_t c = 0; c < nCols; ++c) {
    const int32_t* s = cols + c * KT;
    // every KF-subset of the KT vertices, positions ascending
    std::vector<int> p(KF);
    for (int i = 0; i < KF; ++i) p[i] = i;
    for (;;) {
      Key k;
      for (int i = 0; i < KF; ++i) k[i] = s[p[i]];
      lists[row_id(k)].push_back(int32_t(c));
      int i = KF - 1;
      while (i >= 0 && p[i] == KT - KF + i) --i;
      if (i < 0) break;
      ++p[i];
      for (int j = i + 1; j < KF; ++j) p[j] = p[j - 1] + 1;
    }
  }
  C.off.assign(nRows + 1, 0);
  for (int64_t r = 0; r < nRows; ++r) {
    C.off[r + 1] = C.off[r] + int64_t(lists[r].size());
    C.idx.insert(C.idx.end(), lists[r].begin(), lists[r].end());
  }
}
extern "C" {
void* go_coboundary(int dim, int from, int to, int64_t nV, int64_t nT, const int32_t* T) {
  const int D = dim + 1;
  SubSimplices* R = from == 2 ? enumerate_sub<2>(D, nV, nT, T) : enumerate_sub<3>(D, nV, nT, T);
  Cobound* C = new Cobound;
  if (to == D) {
    if (from == 2) cobound_fill<2>(*C, R->list, D, nT, T); else cobound_fill<3>(*C, R->list, D, nT, T);
  } else {  // to == 3 < D: the containing simplices are the triangles of F
    SubSimplices* F = enumerate_sub<3>(D, nV, nT, T);
    cobound_fill<2>(*C, R->list, 3, int64_t(F->list.size()) / 3, F->list.data());
    delete F;
  }
  delete R;
  return C;
}
int64_t go_cob_rows(void* h) { return int64_t(static_cast<Cobound*>(h)->off.size()) - 1; }
const int64_t* go_cob_off(void* h) { return static_cast<Cobound*>(h)->off.data(); }
const int32_t* go_cob_idx(void* h) { return static_cast<Cobound*>(h)->idx.data(); }
void go_cob_release(void* h) { delete static_cast<Cobound*>(h); }

// ---- brute-force enumeration (tiny meshes; pins the routines above) ------------------------------
// Membership scans straight from the definitions; no sorting, no transposition.
static bool contains(const int32_t* r, int D, int32_t v) {
  for (int k = 0; k < D; ++k)
    if (r[k] == v) return true;
  return false;
}
// VT(v) by scanning every simplex: O(nV*nT*D). off has nV+1 entries, idx D*nT.
void go_brute_vt(int dim, int64_t nV, int64_t nT, const int32_t* T, int64_t* off, int32_t* idx) {
  const int D = dim + 1;
  int64_t o = 0;
  off[0] = 0;
  for (int64_t v = 0; v < nV; ++v) {
    for (int64_t t = 0; t < nT; ++t)
      if (contains(T + t * D, D, int32_t(v))) idx[o++] = int32_t(t);
    off[v + 1] = o;
  }
}
// VV(v) by testing every pair (v,u) against every simplex: O(nV^2*nT*D). idx capacity: D*(D-1)*nT.
void go_brute_vv(int dim, int64_t nV, int64_t nT, const int32_t* T, int64_t* off, int32_t* idx) {
  const int D = dim + 1;
  int64_t o = 0;
  off[0] = 0;
  for (int64_t v = 0; v < nV; ++v) {
    for (int64_t u = 0; u < nV; ++u) {
      if (u == v) continue;
      bool adj = false;
      for (int64_t t = 0; t < nT && !adj; ++t) adj = contains(T + t * D, D, int32_t(v)) && contains(T + t * D, D, int32_t(u));
      if (adj) idx[o++] = int32_t(u);
    }
    off[v + 1] = o;
  }
}
// TT by testing every ordered pair of simplices: O(nT^2*D^2). Returns -4 if some facet has > 2 cofaces.
int go_brute_tt(int dim, int64_t nT, const int32_t* T, int32_t* tt) {
  const int D = dim + 1;
  for (int64_t t = 0; t < nT; ++t)
    for (int k = 0; k < D; ++k) {
      int32_t found = -1;
      for (int64_t s = 0; s < nT; ++s) {
        if (s == t) continue;
        bool all = true;
        for (int j = 0; j < D && all; ++j)
          if (j != k) all = contains(T + s * D, D, T[t * D + j]);
        if (all) {
          if (found >= 0) return GO_NONMANIFOLD;
          found = int32_t(s);
        }
      }
      tt[t * D + k] = found;
    }
  return GO_OK;
}

}  // extern "C"
