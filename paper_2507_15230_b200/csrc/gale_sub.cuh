// gale_sub.cuh — edges and triangles: the sorted lists E and F with their interval
// arrays I_E / I_F, built at initialization only when asked for (the paper's preconditioning),
// and the coboundary relations VE and VF of a cluster batch (Table 1 :53-58; DiscreteGradient
// needs VE, VF, VT, :307).
//
// Layout. A sub-simplex is internal to the segment of its lowest vertex, and the lists are
// sorted by vertex indices, so the edges with lowest vertex a are the contiguous ids
// [e_first[a], e_first[a+1]) and only their upper vertex is stored (e_hi); likewise the triangles with
// lowest vertex a are [f_first[a], f_first[a+1]) and (second, third) vertex are stored (f_bc). An id is
// found by a binary search bounded by the interval array, exactly the paper's look-up (:186-192).
//
// VE(v)[i] is the edge between v and VV(v)[i]: edges below v's own block ascend with the lower
// neighbour, v's own block ascends with the upper neighbour — the order of the sorted VV row. So VE is a
// map over the VV rows the batch kernel has just written. VF(v) = the distinct triangles of the simplices
// of VT(v) that contain v, ids ascending: one warp per vertex sorts the candidates in shared memory.
#pragma once
#include <cuda_runtime.h>
#include <limits.h>
#include <stdint.h>

#include "gale_init.cuh"
#include "gale_kernels.cuh"

namespace gale {
namespace sub {

struct SubIndex {               // all DEVICE, owned by the library
  const int32_t* e_first;       // [nV+1] I_E per vertex
  const int32_t* e_hi;          // [nE]   upper vertex of every edge
  const int32_t* f_first;       // [nV+1] I_F per vertex
  const int2* f_bc;             // [nF]   second and third vertex of every triangle
  const int32_t* cl_off;        // [nC+1] I_V: first vertex of every cluster
};

// ---- E from VV rows ----------------------------------------------------------------------------------
// rows [0, n_rows) of a batch whose vertices are consecutive per cluster; one thread per row.
// COUNT: deg_hi[v] = number of neighbours above v; else e_hi[e_first[v] + j] = j-th neighbour above v.
struct BatchRows {
  int n_clusters;
  int row_base[kMaxBatch + 1];  // first row of cluster slot i in the batch (+ total)
  int cluster[kMaxBatch];
};
__device__ __forceinline__ int row_vertex(const BatchRows& B, const int32_t* cl_off, int r) {
  int lo = 0, hi = B.n_clusters;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (B.row_base[mid] <= r) lo = mid; else hi = mid;
  }
  return cl_off[B.cluster[lo]] + (r - B.row_base[lo]);
}
template <bool COUNT>
__global__ void k_upper_edges(const __grid_constant__ BatchRows B, const int32_t* __restrict__ cl_off,
                              const int32_t* __restrict__ vv_off, const int32_t* __restrict__ vv_idx,
                              int32_t* deg_or_first, int32_t* e_hi) {
  const int r = B.row_base[0] + blockIdx.x * blockDim.x + threadIdx.x;  // rows of this launch: [row_base[0], row_base[n])
  if (r >= B.row_base[B.n_clusters]) return;
  const int v = row_vertex(B, cl_off, r);
  const int a = vv_off[r], b = vv_off[r + 1];
  int lo = a, hi = b;  // first entry above v (the row is ascending)
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (vv_idx[mid] < v) lo = mid + 1; else hi = mid;
  }
  if (COUNT) {
    deg_or_first[v] = b - lo;
  } else {
    int32_t* out = e_hi + deg_or_first[v];
    for (int i = lo; i < b; ++i) out[i - lo] = vv_idx[i];
  }
}

// ---- F from the facet groups of the vertices ----------------------------------------------------------
// The triangles with lowest vertex a are the facets (a, x, y) of the simplices of a's run (three each)
// and the facets opposite the lowest vertex of the simplices whose second vertex is a (one each). One warp
// per vertex collects them as 64-bit keys (x, y), sorts them in shared memory and drops the duplicates.
// COUNT: cnt[a] = distinct triangles; else f_bc[f_first[a] + j] = j-th. Dynamic shared memory:
// (warps per block) * cap * 8 bytes, cap = power of two >= the largest group.
__device__ __forceinline__ void warp_bitonic64(unsigned long long* a, int n2, int lane) {
  for (int k = 2; k <= n2; k <<= 1)
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int i = lane; i < n2; i += 32) {
        const int p = i ^ j;
        if (p > i) {
          const unsigned long long x = a[i], y = a[p];
          const bool up = (i & k) == 0;
          if ((x > y) == up) { a[i] = y; a[p] = x; }
        }
      }
      __syncwarp();
    }
}
template <bool COUNT>
__global__ void k_triangles(const int32_t* __restrict__ T, const int32_t* __restrict__ first_tet,
                            const int32_t* __restrict__ opp_first, const int32_t* __restrict__ opp_perm, int nV, int cap,
                            int32_t* cnt_or_first, int2* f_bc) {
  extern __shared__ unsigned long long shk[];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int a = blockIdx.x * (blockDim.x >> 5) + w;
  if (a >= nV) return;
  unsigned long long* keys = shk + (size_t)w * cap;
  const int r0 = first_tet[a], r1 = first_tet[a + 1], o0 = opp_first[a], o1 = opp_first[a + 1];
  const int n = 3 * (r1 - r0) + (o1 - o0);
  const int n2 = init::pow2_ceil(n < 1 ? 1 : n);
  const int4* T4 = reinterpret_cast<const int4*>(T);
  auto key = [](int x, int y) { return ((unsigned long long)(unsigned)x << 32) | (unsigned)y; };
  for (int i = lane; i < n2; i += 32) {
    unsigned long long k = ~0ull;
    if (i < 3 * (r1 - r0)) {
      const int4 q = __ldg(T4 + r0 + i / 3);
      const int f = i % 3;  // (b,c), (b,d), (c,d)
      k = f == 0 ? key(q.y, q.z) : (f == 1 ? key(q.y, q.w) : key(q.z, q.w));
    } else if (i < n) {
      const int4 q = __ldg(T4 + __ldg(opp_perm + o0 + (i - 3 * (r1 - r0))));
      k = key(q.z, q.w);
    }
    keys[i] = k;
  }
  __syncwarp();
  warp_bitonic64(keys, n2, lane);
  int base = 0;
  for (int i0 = 0; i0 < n2; i0 += 32) {  // heads in order
    const int i = i0 + lane;
    const bool head = i < n2 && keys[i] != ~0ull && (i == 0 || keys[i] != keys[i - 1]);
    const unsigned m = __ballot_sync(0xFFFFFFFFu, head);
    if (!COUNT && head) {
      const unsigned long long k = keys[i];
      f_bc[cnt_or_first[a] + base + __popc(m & ((1u << lane) - 1u))] = make_int2((int)(k >> 32), (int)(k & 0xFFFFFFFFu));
    }
    base += __popc(m);
  }
  if (COUNT && lane == 0) cnt_or_first[a] = base;
}

// ---- VE of a batch: a map over its VV rows -------------------------------------------------------------
__global__ void k_ve(const __grid_constant__ BatchRows B, const SubIndex X, const int32_t* __restrict__ vv_off,
                     const int32_t* __restrict__ vv_idx, int32_t* ve_idx) {
  const int r = B.row_base[0] + blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= B.row_base[B.n_clusters]) return;
  const int v = row_vertex(B, X.cl_off, r);
  const int a = vv_off[r], b = vv_off[r + 1];
  int own = X.e_first[v];
  for (int i = a; i < b; ++i) {
    const int u = vv_idx[i];
    int id;
    if (u < v) {  // the edge is internal to u's segment: look v up among u's upper neighbours
      int lo = X.e_first[u], hi = X.e_first[u + 1];
      while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (X.e_hi[mid] < v) lo = mid + 1; else hi = mid;
      }
      id = lo;
    } else {
      id = own++;  // v's own block, in the order of its upper neighbours
    }
    GALE_ST(ve_idx + i, id);
  }
}

// largest row length of a CSR (sizes the candidate buffers of k_vf)
__global__ void k_max_row(const int32_t* __restrict__ off, int n_rows, int* out) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  int d = r < n_rows ? off[r + 1] - off[r] : 0;
#pragma unroll
  for (int k = 16; k > 0; k >>= 1) d = max(d, __shfl_xor_sync(0xFFFFFFFFu, d, k));
  if ((threadIdx.x & 31) == 0 && d > 0) atomicMax(out, d);
}

// ---- VF of a batch -------------------------------------------------------------------------------------
// One block per tile (its rows), one warp per vertex in turn, over the VT rows the batch kernel has just
// written. Candidates: for every simplex of VT(v) the three triangles that contain v; id of a triangle
// (a, b, c) = position of (b, c) in a's block of F. COUNT (sizing at create): stats[tile] = entries of the
// tile, nothing else is written. Dynamic shared memory (ints): 2 * ((rows + 4) & ~3) for the degrees +
// warps * cap for the candidates + rows * cap for the rows' results (not in count mode), cap = power of
// two >= 3 * the largest |VT(v)|.
struct VFParams {
  int n_clusters;
  int total_rows, total_vf;         // terminal offset
  int tile_prefix[kMaxBatch + 1];
  int cluster[kMaxBatch];
  int row_base[kMaxBatch];          // first VT row of slot i in the batch
  int vf_base[kMaxBatch];           // first VF entry of slot i in the batch
};
__device__ __forceinline__ int tri_id(const SubIndex& X, int a, int b, int c) {
  int lo = X.f_first[a], hi = X.f_first[a + 1];
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    const int2 q = X.f_bc[mid];
    if (q.x < b || (q.x == b && q.y < c)) lo = mid + 1; else hi = mid;
  }
  return lo;
}
__device__ __forceinline__ void warp_bitonic32(int32_t* a, int n2, int lane) {
  for (int k = 2; k <= n2; k <<= 1)
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int i = lane; i < n2; i += 32) {
        const int p = i ^ j;
        if (p > i) {
          const int x = a[i], y = a[p];
          const bool up = (i & k) == 0;
          if ((x > y) == up) { a[i] = y; a[p] = x; }
        }
      }
      __syncwarp();
    }
}
template <bool COUNT>
__global__ void k_vf(const DeviceMesh M, const SubIndex X, const __grid_constant__ VFParams P, int cap,
                     const int32_t* __restrict__ tile_vf_rel, const int32_t* __restrict__ vt_off,
                     const int32_t* __restrict__ vt_idx, int32_t* vf_off, int32_t* vf_idx, int32_t* stats) {
  extern __shared__ int32_t shv[];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  if (!COUNT && blockIdx.x == 0 && threadIdx.x == 0) { vf_off[0] = 0; vf_off[P.total_rows] = P.total_vf; }  // every launch of a batch writes the same two values
  if ((int)blockIdx.x >= P.tile_prefix[P.n_clusters]) return;
  int slot;
  {
    int lo = 0, hi = P.n_clusters;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (P.tile_prefix[mid] <= (int)blockIdx.x) lo = mid; else hi = mid;
    }
    slot = lo;
  }
  const int tile = M.cluster_tile_begin[P.cluster[slot]] + ((int)blockIdx.x - P.tile_prefix[slot]);
  const int nrows = M.tiles[tile].nrows, v_lo = M.tiles[tile].v_lo;
  const int row0 = P.row_base[slot] + M.tiles[tile].row_rel;
  // shared memory: deg[nrows+1] | nlow[nrows] | cand[warps][cap] | keep[nrows][cap] (not in count mode)
  const int pad = (nrows + 4) & ~3;
  int32_t* deg = shv;
  int32_t* nlow = shv + pad;
  int32_t* cand = shv + 2 * pad + (size_t)w * cap;
  int32_t* keep = shv + 2 * pad + (size_t)nw * cap;
  const int4* T4 = reinterpret_cast<const int4*>(M.T);
  // The triangles that have v as their LOWEST vertex are v's own block of F: contiguous ids, no look-up.
  // The others lie in the blocks of lower vertices (smaller ids): they come from the simplices of VT(v) in
  // which v is not the lowest vertex — each such triangle is found in at most two of them — and are
  // looked up, sorted and de-duplicated by the warp.
  for (int r = w; r < nrows; r += nw) {
    const int v = v_lo + r;
    const int t0 = vt_off[row0 + r], t1 = vt_off[row0 + r + 1];
    const int n = min(3 * (t1 - t0), cap);
    int nc = 0;  // candidates kept so far (compacted: the sort below is as small as the looked-up part)
    for (int i0 = 0; i0 < n; i0 += 32) {
      const int i = i0 + lane;
      int id = INT_MAX;
      if (i < n) {
        const int4 q = __ldg(T4 + vt_idx[t0 + i / 3]);
        if (q.x != v) {                                      // v is not the lowest vertex of this simplex
          const int s[4] = {q.x, q.y, q.z, q.w};
          int o[3] = {0, 0, 0}, m = 0;
#pragma unroll
          for (int k = 0; k < 4; ++k)
            if (s[k] != v && m < 3) o[m++] = s[k];          // the three other vertices, ascending
          const int f = i % 3;                              // drop one of them: (v, o1, o2), (v, o0, o2), (v, o0, o1)
          const int x = f == 0 ? o[1] : o[0], y = f == 2 ? o[1] : o[2];
          if (x < v) {                                       // else v is the lowest vertex of the triangle: own block
            int a = x, b = v, c = y;                         // x < v, x < y: sort (v, y)
            if (b > c) { const int tt = b; b = c; c = tt; }
            id = tri_id(X, a, b, c);
          }
        }
      }
      const unsigned mk = __ballot_sync(0xFFFFFFFFu, id != INT_MAX);
      if (id != INT_MAX) cand[nc + __popc(mk & ((1u << lane) - 1u))] = id;
      nc += __popc(mk);
    }
    const int n2 = init::pow2_ceil(nc < 1 ? 1 : nc);
    for (int i = nc + lane; i < n2; i += 32) cand[i] = INT_MAX;
    __syncwarp();
    warp_bitonic32(cand, n2, lane);
    int base = 0;
    for (int i0 = 0; i0 < n2; i0 += 32) {
      const int i = i0 + lane;
      const bool head = i < n2 && cand[i] != INT_MAX && (i == 0 || cand[i] != cand[i - 1]);
      const unsigned m = __ballot_sync(0xFFFFFFFFu, head);
      if (!COUNT && head) keep[(size_t)r * cap + base + __popc(m & ((1u << lane) - 1u))] = cand[i];
      base += __popc(m);
    }
    __syncwarp();
    if (lane == 0) { nlow[r] = base; deg[r] = base + (X.f_first[v + 1] - X.f_first[v]); }
  }
  __syncthreads();
  if (threadIdx.x == 0) {  // a tile has few rows: serial exclusive scan
    int acc = COUNT ? 0 : P.vf_base[slot] + tile_vf_rel[tile];
    for (int r = 0; r < nrows; ++r) { const int d = deg[r]; deg[r] = acc; acc += d; }
    deg[nrows] = acc;
    if (COUNT) stats[tile] = acc;
  }
  __syncthreads();
  if constexpr (!COUNT) {
  for (int r = threadIdx.x; r < nrows; r += blockDim.x) vf_off[row0 + r] = deg[r];
  for (int r = w; r < nrows; r += nw) {  // write-out, one warp per row: the looked-up ids, then the own block
    const int nl = nlow[r], tot = deg[r + 1] - deg[r], own0 = X.f_first[v_lo + r];
    int32_t* out = vf_idx + deg[r];
    for (int i = lane; i < tot; i += 32) GALE_ST(out + i, i < nl ? keep[(size_t)r * cap + i] : own0 + (i - nl));
  }
  }
}

// ---- EF, ET, FT of a batch (PAPER.md:49, Table 1; the MS-complex set, :309) ----------------------------
// Rows = the edges (E..) / triangles (F..) internal to the requested clusters, i.e. the blocks of E / F of
// their vertices; the rows of a tile are contiguous ids. One block per tile, one warp per vertex a: the
// simplices of VT(a) (just written by the batch kernel) are held in shared memory; row (a, b) of ET = those
// that contain b, row (a, b, c) of FT = those that contain b and c — a ballot per 32 simplices, in VT's
// ascending order; row (a, b) of EF = the triangles (a, b, x) of those simplices, looked up in F, sorted
// and de-duplicated by the warp. COUNT (sizing at create): stats[tile] = entries of the tile.
// Dynamic shared memory (ints): rows_cap + 4 (row counts -> offsets) | ((nrows + 4) & ~3) (vertex totals) |
// warps * star_cap * 4 (the stars) | warps * 64 (EF candidates).
enum { COB_ET = 0, COB_FT = 1, COB_EF = 2 };
struct CobParams {
  int n_clusters;
  int total_rows, total_nnz;        // terminal offset
  int tile_prefix[kMaxBatch + 1];
  int cluster[kMaxBatch];
  int vt_row_base[kMaxBatch];       // first VT row of slot i in the batch
  int row_base[kMaxBatch];          // first edge / triangle row of slot i in the batch
  int nnz_base[kMaxBatch];          // first entry of slot i in the batch
};
template <int KIND, bool COUNT>
__global__ void k_cob(const DeviceMesh M, const SubIndex X, const __grid_constant__ CobParams P, int rows_cap, int star_cap,
                      const int32_t* __restrict__ tile_rel, const int32_t* __restrict__ vt_off,
                      const int32_t* __restrict__ vt_idx, int32_t* out_off, int32_t* out_idx, int32_t* stats) {
  extern __shared__ int32_t shc[];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  if (!COUNT && blockIdx.x == 0 && threadIdx.x == 0) { out_off[0] = 0; out_off[P.total_rows] = P.total_nnz; }
  if ((int)blockIdx.x >= P.tile_prefix[P.n_clusters]) return;
  int slot;
  {
    int lo = 0, hi = P.n_clusters;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (P.tile_prefix[mid] <= (int)blockIdx.x) lo = mid; else hi = mid;
    }
    slot = lo;
  }
  const int tile = M.cluster_tile_begin[P.cluster[slot]] + ((int)blockIdx.x - P.tile_prefix[slot]);
  const int nrows = M.tiles[tile].nrows, v_lo = M.tiles[tile].v_lo;
  const int c_lo = v_lo - M.tiles[tile].row_rel;
  const int32_t* first = KIND == COB_FT ? X.f_first : X.e_first;   // interval array of the ROW list
  const int r_tile0 = first[v_lo], r_tile1 = first[v_lo + nrows];   // the tile's rows: contiguous ids
  const int n_tile_rows = min(r_tile1 - r_tile0, rows_cap);
  const int vrow0 = P.vt_row_base[slot] + M.tiles[tile].row_rel;
  int32_t* rcnt = shc;                                   // [rows_cap + 1] counts, then offsets
  int32_t* vtot = shc + ((rows_cap + 4) & ~3);           // [nrows + 1]
  int4* star = reinterpret_cast<int4*>(vtot + ((nrows + 4) & ~3)) + (size_t)w * star_cap;
  int32_t* cand = reinterpret_cast<int32_t*>(reinterpret_cast<int4*>(vtot + ((nrows + 4) & ~3)) + (size_t)nw * star_cap) + w * 64;
  const int4* T4 = reinterpret_cast<const int4*>(M.T);
  for (int pass = 0; pass < (COUNT ? 1 : 2); ++pass) {
    for (int r = w; r < nrows; r += nw) {
      const int a = v_lo + r;
      const int t0 = vt_off[vrow0 + r];
      const int deg = min(vt_off[vrow0 + r + 1] - t0, star_cap);
      for (int i = lane; i < deg; i += 32) star[i] = __ldg(T4 + vt_idx[t0 + i]);
      __syncwarp();
      int tot = 0;
      const int j0 = first[a], j1 = first[a + 1];
      for (int j = j0; j < j1; ++j) {
        const int jr = j - r_tile0;                       // row inside the tile
        int b, c = -1;
        if (KIND == COB_FT) { const int2 q = X.f_bc[j]; b = q.x; c = q.y; } else { b = X.e_hi[j]; }
        const int wbase = (pass == 1 && jr < rows_cap) ? rcnt[jr] : 0;
        int cnt = 0;
        if (KIND != COB_EF) {
          for (int i0 = 0; i0 < deg; i0 += 32) {
            const int i = i0 + lane;
            bool hit = false;
            if (i < deg) {
              const int4 q = star[i];
              const bool hb = q.x == b || q.y == b || q.z == b || q.w == b;
              hit = KIND == COB_FT ? (hb && (q.x == c || q.y == c || q.z == c || q.w == c)) : hb;
            }
            const unsigned m = __ballot_sync(0xFFFFFFFFu, hit);
            if (pass == 1 && hit) GALE_ST(out_idx + wbase + cnt + __popc(m & ((1u << lane) - 1u)), vt_idx[t0 + i]);
            cnt += __popc(m);
          }
        } else {
          int nc = 0;                                     // triangles (a, b, x) of the simplices that contain b
          for (int i0 = 0; i0 < deg; i0 += 32) {
            const int i = i0 + lane;
            int id0 = INT_MAX, id1 = INT_MAX;
            if (i < deg) {
              const int4 q = star[i];
              const int s[4] = {q.x, q.y, q.z, q.w};
              if (s[0] == b || s[1] == b || s[2] == b || s[3] == b) {
                int o[2] = {0, 0}, mm = 0;
#pragma unroll
                for (int k = 0; k < 4; ++k)
                  if (s[k] != a && s[k] != b && mm < 2) o[mm++] = s[k];
#pragma unroll
                for (int u = 0; u < 2; ++u) {               // sort (a, b, x): a < b
                  const int x = o[u];
                  const int p0 = x < a ? x : a, p2 = x > b ? x : b, p1 = a + b + x - p0 - p2;
                  (u == 0 ? id0 : id1) = tri_id(X, p0, p1, p2);
                }
              }
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
              const int id = u == 0 ? id0 : id1;
              const unsigned m = __ballot_sync(0xFFFFFFFFu, id != INT_MAX);
              if (id != INT_MAX && nc + __popc(m & ((1u << lane) - 1u)) < 64) cand[nc + __popc(m & ((1u << lane) - 1u))] = id;
              nc = min(64, nc + __popc(m));
            }
          }
          const int n2 = init::pow2_ceil(nc < 1 ? 1 : nc);
          for (int i = nc + lane; i < n2; i += 32) cand[i] = INT_MAX;
          __syncwarp();
          warp_bitonic32(cand, n2, lane);
          for (int i0 = 0; i0 < n2; i0 += 32) {
            const int i = i0 + lane;
            const bool head = i < n2 && cand[i] != INT_MAX && (i == 0 || cand[i] != cand[i - 1]);
            const unsigned m = __ballot_sync(0xFFFFFFFFu, head);
            if (pass == 1 && head) GALE_ST(out_idx + wbase + cnt + __popc(m & ((1u << lane) - 1u)), cand[i]);
            cnt += __popc(m);
          }
          __syncwarp();
        }
        if (pass == 0 && lane == 0 && jr < rows_cap) rcnt[jr] = cnt;
        tot += cnt;
      }
      if (pass == 0 && lane == 0) vtot[r] = tot;
      __syncwarp();
    }
    __syncthreads();
    if (pass == 0) {
      if (threadIdx.x == 0) {  // serial exclusive scan over the tile's rows (a few hundred)
        int acc = COUNT ? 0 : P.nnz_base[slot] + tile_rel[tile];
        for (int j = 0; j < n_tile_rows; ++j) { const int d = rcnt[j]; rcnt[j] = acc; acc += d; }
        rcnt[n_tile_rows] = acc;
        if (COUNT) stats[tile] = acc;
      }
      __syncthreads();
      if (!COUNT) {
        const int orow0 = P.row_base[slot] + (r_tile0 - first[c_lo]);
        for (int j = threadIdx.x; j < n_tile_rows; j += blockDim.x) out_off[orow0 + j] = rcnt[j];
      }
    }
  }
}

}  // namespace sub
}  // namespace gale
