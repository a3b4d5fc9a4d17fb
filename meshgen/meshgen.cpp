// meshgen — seeded synthetic simplicial-mesh generator (host C++, C ABI).
//
// This module only *builds inputs*: Kuhn-triangulated grids, jitter / warp of
// coordinates, a seeded vertex permutation, Morton and PR-octree vertex
// clustering ("PR octree ... maximum number of vertices per leaf"),
// renumbering and canonicalisation (SURVEY.md §8(c) input contract C1-C3).
// It holds none of the method's arithmetic (no VT / VV / TT) and is the one
// piece of code that serves both the CPU oracle and the CUDA path.
//
// Recipe and seeds: SURVEY.md §8(d); restated in DESIGN.md §Input recipe.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>

namespace {

inline uint64_t splitmix64(uint64_t x) {
  x += 0x9E3779B97F4A7C15ull;
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
  return x ^ (x >> 31);
}
// counter-based uniform in [0,1) with 24 random bits (exact in float32)
inline float u01(uint64_t seed, uint64_t i) {
  return float(splitmix64(seed + i * 0x9E3779B97F4A7C15ull) >> 40) * (1.0f / 16777216.0f);
}
inline uint64_t rnd64(uint64_t seed, uint64_t i) {
  return splitmix64(seed + i * 0x9E3779B97F4A7C15ull);
}

inline uint64_t spread3(uint64_t v) {  // 20 bits -> every third bit
  v &= 0xFFFFFull;
  v = (v | (v << 32)) & 0x1F00000000FFFFull;
  v = (v | (v << 16)) & 0x1F0000FF0000FFull;
  v = (v | (v << 8)) & 0x100F00F00F00F00Full;
  v = (v | (v << 4)) & 0x10C30C30C30C30C3ull;
  v = (v | (v << 2)) & 0x1249249249249249ull;
  return v;
}
inline uint64_t spread2(uint64_t v) {  // 20 bits -> every second bit
  v &= 0xFFFFFull;
  v = (v | (v << 16)) & 0x0000FFFF0000FFFFull;
  v = (v | (v << 8)) & 0x00FF00FF00FF00FFull;
  v = (v | (v << 4)) & 0x0F0F0F0F0F0F0F0Full;
  v = (v | (v << 2)) & 0x3333333333333333ull;
  v = (v | (v << 1)) & 0x5555555555555555ull;
  return v;
}
inline uint64_t morton(int dim, uint32_t x, uint32_t y, uint32_t z) {
  return dim == 3 ? (spread3(x) | (spread3(y) << 1) | (spread3(z) << 2))
                  : (spread2(x) | (spread2(y) << 1));
}

}  // namespace

extern "C" {

// Number of vertices / simplices of an n^dim Kuhn grid.
int64_t mg_grid_num_vertices(int dim, int n) {
  int64_t v = 1;
  for (int i = 0; i < dim; ++i) v *= n;
  return v;
}
int64_t mg_grid_num_simplices(int dim, int n) {
  int64_t m = n - 1, c = 1;
  for (int i = 0; i < dim; ++i) c *= m;
  return c * (dim == 3 ? 6 : 2);
}

// Kuhn (Freudenthal) triangulation: each cube -> one simplex per permutation pi of the
// axes, p0 = corner, p_{i+1} = p_i + e_{pi(i)}; all share the main diagonal.
// Vertex id = x + n*(y + n*z). Rows are written unsorted, in cube order.
void mg_kuhn_grid(int dim, int n, int32_t* T) {
  const int64_t m = n - 1;
  int64_t o = 0;
  if (dim == 3) {
    static const int P[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
    const int64_t st[3] = {1, n, int64_t(n) * n};
    for (int64_t z = 0; z < m; ++z)
      for (int64_t y = 0; y < m; ++y)
        for (int64_t x = 0; x < m; ++x) {
          const int64_t c = x + n * (y + n * z);
          for (int p = 0; p < 6; ++p) {
            int64_t v = c;
            T[o++] = int32_t(v);
            for (int i = 0; i < 3; ++i) {
              v += st[P[p][i]];
              T[o++] = int32_t(v);
            }
          }
        }
  } else {
    for (int64_t y = 0; y < m; ++y)
      for (int64_t x = 0; x < m; ++x) {
        const int64_t c = x + n * y;
        T[o++] = int32_t(c); T[o++] = int32_t(c + 1); T[o++] = int32_t(c + 1 + n);
        T[o++] = int32_t(c); T[o++] = int32_t(c + n); T[o++] = int32_t(c + 1 + n);
      }
  }
}

// coords[v*dim + a] = grid position + (u - 0.5)*0.4  (jitter +-0.2 cell), float32.
// warp != 0: normalise each axis to [0,1] over the grid extent incl. jitter margin, then x -> x^3.
void mg_coords(int dim, int n, uint64_t seed, int warp, float* xyz) {
  const int64_t nV = mg_grid_num_vertices(dim, n);
  for (int64_t v = 0; v < nV; ++v) {
    int64_t r = v;
    for (int a = 0; a < dim; ++a) {
      const int64_t g = r % n;
      r /= n;
      double c = double(g) + (double(u01(seed, uint64_t(v) * 3 + a)) - 0.5) * 0.4;
      if (warp) {
        double t = (c + 0.2) / (double(n - 1) + 0.4);
        t = std::min(1.0, std::max(0.0, t));
        c = t * t * t;
      }
      xyz[v * dim + a] = float(c);
    }
  }
}

void mg_scalar(int64_t nV, uint64_t seed, float* f) {
  for (int64_t v = 0; v < nV; ++v) f[v] = u01(seed, uint64_t(v));
}

// Fisher-Yates with the counter-based generator: perm[i] = new id of old vertex i.
void mg_permutation(int64_t nV, uint64_t seed, int32_t* perm) {
  for (int64_t i = 0; i < nV; ++i) perm[i] = int32_t(i);
  for (int64_t i = nV - 1; i > 0; --i) {
    const uint64_t j = rnd64(seed, uint64_t(i)) % uint64_t(i + 1);
    std::swap(perm[i], perm[j]);
  }
}

// Morton clustering of a regular grid: order[rank] = grid vertex id in Morton order of its
// integer grid position (x lowest bit); clusters = aligned block^dim cells, ordered by the
// Morton code of the block. Returns the number of clusters; offsets has that many + 1.
// Requires block | n and n/block, block powers of two.
int32_t mg_morton_clusters(int dim, int n, int block, int32_t* order, int32_t* offsets) {
  const int64_t nV = mg_grid_num_vertices(dim, n);
  std::vector<uint64_t> key(nV);
  for (int64_t v = 0; v < nV; ++v) {
    const uint32_t x = uint32_t(v % n), y = uint32_t((v / n) % n), z = dim == 3 ? uint32_t(v / (int64_t(n) * n)) : 0u;
    key[v] = morton(dim, x, y, z);
  }
  std::vector<int32_t> idx(nV);
  std::iota(idx.begin(), idx.end(), 0);
  std::sort(idx.begin(), idx.end(), [&](int32_t a, int32_t b) { return key[a] < key[b]; });
  std::memcpy(order, idx.data(), sizeof(int32_t) * nV);
  int64_t per = 1;
  for (int i = 0; i < dim; ++i) per *= block;
  const int64_t nC = nV / per;
  for (int64_t c = 0; c <= nC; ++c) offsets[c] = int32_t(c * per);
  return int32_t(nC);
}

// PR-octree (quadtree in 2-D) clustering. Bounding cube of the coordinates (side = largest
// extent), coordinates quantised to 2^20 cells per axis, a node holding more than `capacity`
// points splits at its centre into 2^dim children visited in Morton order (x lowest); a point on
// a split plane goes to the upper child (floor quantisation); empty leaves are dropped; depth cap
// 20; inside a leaf vertices are ordered by Morton code, ties by previous id.
// order[rank] = old vertex id; offsets: leaf boundaries. Returns the number of leaves
// (offsets must have room for nV + 1 entries in the worst case).
int32_t mg_octree_clusters(int dim, int64_t nV, const float* xyz, int32_t capacity, int32_t* order,
                           int32_t* offsets) {
  double lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
  for (int a = 0; a < dim; ++a) lo[a] = hi[a] = xyz[a];
  for (int64_t v = 0; v < nV; ++v)
    for (int a = 0; a < dim; ++a) {
      lo[a] = std::min(lo[a], double(xyz[v * dim + a]));
      hi[a] = std::max(hi[a], double(xyz[v * dim + a]));
    }
  double side = 0;
  for (int a = 0; a < dim; ++a) side = std::max(side, hi[a] - lo[a]);
  if (side <= 0) side = 1;
  const double scale = 1048576.0 / side;
  struct KV { uint64_t key; int32_t id; };
  std::vector<KV> kv(nV);
  for (int64_t v = 0; v < nV; ++v) {
    uint32_t q[3] = {0, 0, 0};
    for (int a = 0; a < dim; ++a) {
      double t = std::floor((double(xyz[v * dim + a]) - lo[a]) * scale);
      q[a] = uint32_t(std::min(1048575.0, std::max(0.0, t)));
    }
    kv[v] = {morton(dim, q[0], q[1], q[2]), int32_t(v)};
  }
  std::sort(kv.begin(), kv.end(), [](const KV& a, const KV& b) { return a.key < b.key || (a.key == b.key && a.id < b.id); });
  for (int64_t v = 0; v < nV; ++v) order[v] = kv[v].id;

  // recursive split of [b,e) at `depth` (bits of the key consumed = dim*depth, from the top)
  int32_t nLeaf = 0;
  offsets[0] = 0;
  struct Node { int64_t b, e; int depth; };
  std::vector<Node> stack;
  stack.push_back({0, nV, 0});
  const int fan = 1 << dim;
  while (!stack.empty()) {
    const Node nd = stack.back();
    stack.pop_back();
    if (nd.e == nd.b) continue;
    if (nd.e - nd.b <= capacity || nd.depth >= 20) {
      offsets[++nLeaf] = int32_t(nd.e);
      continue;
    }
    const int shift = dim * (20 - nd.depth - 1);
    // children in Morton order: push in reverse so child 0 is processed first
    int64_t bounds[9];
    bounds[0] = nd.b;
    for (int c = 1; c <= fan; ++c) {
      // first index in [b,e) whose child digit >= c
      int64_t l = bounds[c - 1], r = nd.e;
      while (l < r) {
        const int64_t mid = (l + r) >> 1;
        if (int((kv[mid].key >> shift) & uint64_t(fan - 1)) < c) l = mid + 1; else r = mid;
      }
      bounds[c] = l;
    }
    for (int c = fan - 1; c >= 0; --c) stack.push_back({bounds[c], bounds[c + 1], nd.depth + 1});
  }
  return nLeaf;
}

// Drop a seeded fraction of simplices (perforated mesh). Keeps order; returns the new count.
int64_t mg_drop_simplices(int dim, int64_t nT, int32_t* T, uint64_t seed, double frac) {
  const int D = dim + 1;
  int64_t o = 0;
  for (int64_t t = 0; t < nT; ++t) {
    if (double(u01(seed, uint64_t(t))) < frac) continue;
    if (o != t) std::memcpy(T + o * D, T + t * D, sizeof(int32_t) * D);
    ++o;
  }
  return o;
}

// Renumber vertices (new_id[old]) and canonicalise: every row ascending (C1), rows in
// ascending lexicographic order (C2). Bucket by smallest vertex, then sort each bucket.
// scratch must hold nT*D int32. Result in T.
void mg_renumber_canonicalise(int dim, int64_t nV, int64_t nT, int32_t* T, const int32_t* new_id,
                              int32_t* scratch) {
  const int D = dim + 1;
  std::vector<int64_t> first(nV + 1, 0);
  for (int64_t t = 0; t < nT; ++t) {
    int32_t* r = T + t * D;
    for (int k = 0; k < D; ++k) r[k] = new_id ? new_id[r[k]] : r[k];
    std::sort(r, r + D);
    ++first[r[0] + 1];
  }
  for (int64_t v = 0; v < nV; ++v) first[v + 1] += first[v];
  std::vector<int64_t> cur(first.begin(), first.end() - 1);
  for (int64_t t = 0; t < nT; ++t) {
    const int32_t* r = T + t * D;
    std::memcpy(scratch + cur[r[0]]++ * D, r, sizeof(int32_t) * D);
  }
  // sort inside each bucket (buckets are small: one vertex star)
  if (D == 4) {
    struct R4 { int32_t v[4]; };
    R4* s = reinterpret_cast<R4*>(scratch);
    for (int64_t v = 0; v < nV; ++v)
      std::sort(s + first[v], s + first[v + 1], [](const R4& a, const R4& b) {
        return a.v[1] != b.v[1] ? a.v[1] < b.v[1] : a.v[2] != b.v[2] ? a.v[2] < b.v[2] : a.v[3] < b.v[3];
      });
  } else {
    struct R3 { int32_t v[3]; };
    R3* s = reinterpret_cast<R3*>(scratch);
    for (int64_t v = 0; v < nV; ++v)
      std::sort(s + first[v], s + first[v + 1], [](const R3& a, const R3& b) {
        return a.v[1] != b.v[1] ? a.v[1] < b.v[1] : a.v[2] < b.v[2];
      });
  }
  std::memcpy(T, scratch, sizeof(int32_t) * nT * D);
}

}  // extern "C"
