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

// largest row length of a CSR (sizes the star buffers of k_star)
__global__ void k_max_row(const int32_t* __restrict__ off, int n_rows, int* out) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  int d = r < n_rows ? off[r + 1] - off[r] : 0;
#pragma unroll
  for (int k = 16; k > 0; k >>= 1) d = max(d, __shfl_xor_sync(0xFFFFFFFFu, d, k));
  if ((threadIdx.x & 31) == 0 && d > 0) atomicMax(out, d);
}


// ---- VF, EF, ET, FT of a batch (Table 1; DiscreteGradient :307, the MS-complex set :309) ----
// Rows: VF = the vertices of the requested clusters; ET / EF = the edges, FT = the triangles internal to them,
// i.e. the blocks of E / F of their vertices (the rows of a tile are contiguous ids). Every row of a vertex a
// is a subset of one short, ascending list that belongs to a — its "star":
//   ET (a, b)    = the simplices of VT(a) that contain b;  FT (a, b, c) = those that contain b and c;
//   VF (a)       = the triangles at a: for every lower neighbour x of a (VV(a) ascends, so they come first and
//                  in order) the entries of x's block of F that contain a, then a's own block — ids ascend
//                  and every triangle is met once: no look-up, no sort, no duplicates;
//   EF (a, b)    = the triangles at a that contain b.
// One block per tile, everything flat (one thread per item, no warp-wide loops over short lists):
//   A  one warp per vertex copies its source row into shared memory — the VT entries with the vertices of their
//      simplices (ET, FT) or the VV entries with the F blocks of the lower neighbours (VF, EF) — and the
//      descriptors (e_hi / f_bc) of its rows; all loads independent.
//   B  VF, EF: one thread per (vertex a, lower neighbour x) scans x's block of F and keeps a bit per entry that
//      contains a; a block scan over the pairs places the triangles of every vertex (the own blocks are
//      contiguous ids, so their share of the offsets is a difference of I_F). VF writes them out; EF lists them
//      in shared memory with their vertices above a: the star of a.
//   C  ET, FT, EF: one thread per row scans the star of its vertex and keeps a bit per member (the rows come out
//      sorted for free); sizes = popcounts, block scan, the thread writes the row's offset and entries.
// COUNT (sizing at create): stats[tile] = entries of the tile; VF: *stats_max = the most triangles at a vertex.
enum { COB_ET = 0, COB_FT = 1, COB_EF = 2, COB_VF = 3 };
struct CobParams {
  int n_clusters;
  int total_rows, total_nnz;        // terminal offset
  int uniform_tiles;                // > 0: every cluster of the batch has this many tiles (slot = block / it)
  int tile_prefix[kMaxBatch + 1];
  int cluster[kMaxBatch];
  int src_row_base[kMaxBatch];      // first VT / VV row of slot i in the batch
  int row_base[kMaxBatch];          // first output row of slot i in the batch (VF: its vertex rows)
  int nnz_base[kMaxBatch];          // first entry of slot i in the batch
};
struct StarDims {
  int tv;         // vertices of a tile
  int rows_cap;   // rows of a tile: edges (ET, EF), triangles (FT); VF: 0
  int src_cap;    // entries of the tile's source rows: VT (ET, FT) or VV (EF, VF)
  int W;          // words of a row mask: ceil(largest star / 32); VF: 0
  int Wf;         // EF, VF: words of a pair mask: ceil(longest block of F / 32)
  int fstar_cap;  // EF: triangles at the vertices of a tile
};
struct StarLayout {  // offsets in ints, every section a multiple of 4
  int wsum, soff, rfirst, ofirst, fo, s0, s1, s2, pcnt, pmask, desc, rown, rloc, rmask, fid, ftup, total;
};
__host__ __device__ inline StarLayout make_star_layout(int kind, const StarDims& d) {
  auto pad = [](int n) { return (n + 3) & ~3; };
  const bool from_vt = kind == COB_ET || kind == COB_FT, rows = kind != COB_VF;
  StarLayout L;
  int o = 0;
  L.wsum = o;   o += 32;                    // scratch of the block scans
  L.soff = o;   o += pad(d.tv + 1);         // offsets of the source rows
  L.rfirst = o; o += pad(d.tv + 1);         // I_E / I_F of the tile's vertices (rows)
  L.ofirst = o; o += pad(d.tv + 1);         // I_F of the tile's vertices (EF, VF: own blocks)
  L.fo = o;     o += pad(d.tv + 1);         // EF, VF: first triangle at every vertex, inside the tile
  L.s0 = o;     o += pad(d.src_cap);                                 // simplex ids | first entry of x's F block
  L.s1 = o;     o += from_vt ? 3 * pad(d.src_cap) : pad(d.src_cap);  // their 2nd, 3rd, 4th vertices (one array each: rows of different vertices
                                                                     // read different banks) | length of the block (0: x is not below a)
  L.s2 = o;     o += from_vt ? 0 : pad(d.src_cap);                   // | owner a of the pair
  L.pcnt = o;   o += from_vt ? 0 : pad(d.src_cap + 1);               // hits of the pair, then their prefix
  L.pmask = o;  o += from_vt ? 0 : pad(d.src_cap * d.Wf);
  L.desc = o;   o += rows ? pad(d.rows_cap * (kind == COB_FT ? 2 : 1)) : 0;
  L.rown = o;   o += rows ? pad(d.rows_cap) : 0;                     // vertex of the row
  L.rloc = o;   o += rows ? pad(d.rows_cap + 1) : 0;                 // row sizes, then offsets inside the tile
  L.rmask = o;  o += rows ? pad(d.rows_cap * d.W) : 0;
  L.fid = o;    o += kind == COB_EF ? pad(d.fstar_cap) : 0;          // EF: the triangles at the tile's vertices ...
  L.ftup = o;   o += kind == COB_EF ? 2 * pad(d.fstar_cap) : 0;      // ... and their vertices above a (-1: none)
  L.total = o;
  return L;
}
// In-place exclusive scan of v[0, n) in shared memory by the whole block; v[n] = total (also returned). The
// values must be complete (barrier) before the call; wsum = 32 ints of scratch.
__device__ __forceinline__ int block_scan_smem(int32_t* v, int n, int32_t* wsum) {
  const int tid = threadIdx.x, NT = blockDim.x, lane = tid & 31, w = tid >> 5, nw = NT >> 5;
  const int per = (n + NT - 1) / NT;
  const int j0 = min(tid * per, n), j1 = min(j0 + per, n);
  int sum = 0;
  for (int j = j0; j < j1; ++j) sum += v[j];
  int incl = sum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int y = __shfl_up_sync(0xFFFFFFFFu, incl, d);
    if (lane >= d) incl += y;
  }
  if (lane == 31) wsum[w] = incl;
  __syncthreads();
  int before = 0, total = 0;
  for (int k = 0; k < nw; ++k) { const int t = wsum[k]; if (k < w) before += t; total += t; }
  int acc = before + incl - sum;
  for (int j = j0; j < j1; ++j) { const int c = v[j]; v[j] = acc; acc += c; }
  if (tid == 0) v[n] = total;
  __syncthreads();
  return total;
}
template <int KIND, bool COUNT>
__global__ void __launch_bounds__(256)
k_star(const DeviceMesh M, const SubIndex X, const __grid_constant__ CobParams P, const StarDims Dm, const StarLayout L,
       const int32_t* __restrict__ tile_rel, const int32_t* __restrict__ src_off, const int32_t* __restrict__ src_idx,
       int32_t* out_off, int32_t* out_idx, int32_t* stats, int32_t* stats_max) {
  extern __shared__ __align__(16) int32_t shs[];
  constexpr bool FROM_VT = KIND == COB_ET || KIND == COB_FT, ROWS = KIND != COB_VF;
  const int tid = threadIdx.x, NT = blockDim.x, lane = tid & 31, w = tid >> 5, nw = NT >> 5;
  if (!COUNT && blockIdx.x == 0 && tid == 0) { out_off[0] = 0; out_off[P.total_rows] = P.total_nnz; }  // every launch of a batch writes the same two values
  if ((int)blockIdx.x >= P.tile_prefix[P.n_clusters]) return;
  int slot;
  if (P.uniform_tiles > 0) {  // every cluster of the batch has this many tiles
    slot = (int)blockIdx.x / P.uniform_tiles;
  } else {
    int lo = 0, hi = P.n_clusters;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (P.tile_prefix[mid] <= (int)blockIdx.x) lo = mid; else hi = mid;
    }
    slot = lo;
  }
  const int tile = M.cluster_tile_begin[P.cluster[slot]] + ((int)blockIdx.x - P.tile_prefix[slot]);
  const int nrows = min(M.tiles[tile].nrows, Dm.tv), v_lo = M.tiles[tile].v_lo, row_rel = M.tiles[tile].row_rel;
  const int srow0 = P.src_row_base[slot] + row_rel;
  const int W = Dm.W, Wf = Dm.Wf;
  const int32_t* first = KIND == COB_FT ? X.f_first : X.e_first;  // interval array of the ROW list (not VF)
  int32_t* wsum = shs + L.wsum;
  int32_t* soff = shs + L.soff;
  int32_t* rfirst = shs + L.rfirst;
  int32_t* ofirst = shs + L.ofirst;
  int32_t* fo = shs + L.fo;
  int32_t* sid = shs + L.s0;                                   // ET / FT: simplex ids
  const int sp = (Dm.src_cap + 3) & ~3;
  int32_t* ty = shs + L.s1;                                    // ET / FT: 2nd, 3rd, 4th vertex of those simplices (the lowest is never asked for)
  int32_t* tz = ty + sp;
  int32_t* tw = tz + sp;
  int32_t* nf0 = shs + L.s0;                                   // EF / VF: F block of the lower neighbour x of the pair ...
  int32_t* nlen = shs + L.s1;                                  // ... its length (0: x is not below a) ...
  int32_t* nown = shs + L.s2;                                  // ... and a
  int32_t* pcnt = shs + L.pcnt;
  uint32_t* pmask = reinterpret_cast<uint32_t*>(shs + L.pmask);
  int32_t* desc = shs + L.desc;
  int32_t* rown = shs + L.rown;
  int32_t* rloc = shs + L.rloc;
  uint32_t* rmask = reinterpret_cast<uint32_t*>(shs + L.rmask);
  int32_t* fid = shs + L.fid;
  int32_t* fp1 = shs + L.ftup;                                 // EF: the (up to two) vertices above a of the triangles at a, -1: none
  int32_t* fp2 = fp1 + ((Dm.fstar_cap + 3) & ~3);
  // ---- A1: offsets of the tile's vertices ------------------------------------------------------------------
  for (int r = tid; r <= nrows; r += NT) {
    soff[r] = src_off[srow0 + r];
    if constexpr (ROWS) rfirst[r] = first[v_lo + r];
    if constexpr (!FROM_VT) ofirst[r] = X.f_first[v_lo + r];
  }
  __syncthreads();
  const int s_base = soff[0];
  const int n_src = min(soff[nrows] - s_base, Dm.src_cap);
  const int r_tile0 = ROWS ? rfirst[0] : 0;
  const int n_tile_rows = ROWS ? min(rfirst[nrows] - r_tile0, Dm.rows_cap) : 0;
#if GALE_CHECK_BOUNDS
  // the capacities fixed at create hold for this tile (the clamps above and below never bite)
  if (tid == 0) {
    bool ok = M.tiles[tile].nrows <= Dm.tv && soff[nrows] - s_base <= Dm.src_cap;
    if (ROWS) ok = ok && rfirst[nrows] - r_tile0 <= Dm.rows_cap;
    if (KIND == COB_EF) ok = ok && ofirst[nrows] - ofirst[0] <= Dm.fstar_cap;
    (void)GALE_IN_BOUNDS(M.err, ok);
  }
#endif
  // ---- A2: one warp per vertex: its source row and the descriptors of its rows ---------------------------
  for (int r = w; r < nrows; r += nw) {
    const int a = v_lo + r;
    const int i0 = min(soff[r] - s_base, n_src), i1 = min(soff[r + 1] - s_base, n_src);
    for (int i = i0 + lane; i < i1; i += 32) {
      const int e = src_idx[s_base + i];
      if constexpr (FROM_VT) {
        sid[i] = e;
        const int4 q = __ldg(reinterpret_cast<const int4*>(M.T) + e);
        ty[i] = q.y; tz[i] = q.z; tw[i] = q.w;
      } else {
        int f0 = 0, len = 0;
        if (e < a) { f0 = X.f_first[e]; len = X.f_first[e + 1] - f0; }
        nf0[i] = f0;
        nlen[i] = len;
        nown[i] = r;
      }
    }
    if constexpr (ROWS) {
      const int j0 = min(rfirst[r] - r_tile0, n_tile_rows), j1 = min(rfirst[r + 1] - r_tile0, n_tile_rows);
      for (int j = j0 + lane; j < j1; j += 32) {
        if constexpr (KIND == COB_FT) { const int2 q = X.f_bc[r_tile0 + j]; desc[2 * j] = q.x; desc[2 * j + 1] = q.y; }
        else desc[j] = X.e_hi[r_tile0 + j];
        rown[j] = r;
      }
    }
  }
  __syncthreads();
  const int base0 = COUNT ? 0 : P.nnz_base[slot] + tile_rel[tile];
  // ---- B: the triangles at the tile's vertices (VF, EF) -----------------------------------------------------
  if constexpr (!FROM_VT) {
    for (int i = tid; i < n_src; i += NT) {  // one thread per pair (a, lower neighbour x): a bit per entry of x's block that contains a
      const int len = min(nlen[i], 32 * Wf), f0 = nf0[i], a = v_lo + nown[i];
      (void)GALE_IN_BOUNDS(M.err, nlen[i] <= 32 * Wf && nown[i] >= 0 && nown[i] < nrows);
      int cnt = 0;
      for (int k = 0; k < Wf; ++k) {
        uint32_t bits = 0u;
        const int e1 = min(32, len - 32 * k);
        for (int e = 0; e < e1; ++e) {
          const int2 q = X.f_bc[f0 + 32 * k + e];
          bits |= (uint32_t)(q.x == a || q.y == a) << e;
        }
        pmask[i * Wf + k] = bits;
        cnt += __popc(bits);
      }
      pcnt[i] = cnt;
    }
    __syncthreads();
    block_scan_smem(pcnt, n_src, wsum);
    const int ob = ofirst[0];
    for (int r = tid; r <= nrows; r += NT) fo[r] = pcnt[min(soff[r] - s_base, n_src)] + (ofirst[r] - ob);  // own blocks: contiguous ids
    __syncthreads();
    if constexpr (KIND == COB_VF) {
      if (COUNT) {
        if (tid == 0) stats[tile] = fo[nrows];
        int vmax = 0;
        for (int r = tid; r < nrows; r += NT) vmax = max(vmax, fo[r + 1] - fo[r]);
        if (vmax > 0) atomicMax(stats_max, vmax);
      } else {
        const int orow0 = P.row_base[slot] + row_rel;
        for (int r = tid; r < nrows; r += NT) out_off[orow0 + r] = base0 + fo[r];
      }
    }
    if (!COUNT || KIND == COB_EF) {
      for (int i = tid; i < n_src; i += NT) {  // the pair's triangles, in place
        const int r = nown[i], a = v_lo + r, f0 = nf0[i];
        int pos = fo[r] + (pcnt[i] - pcnt[min(soff[r] - s_base, n_src)]);
        for (int k = 0; k < Wf; ++k) {
          uint32_t bits = pmask[i * Wf + k];
          while (bits) {
            const int j = f0 + 32 * k + __ffs(bits) - 1;
            bits &= bits - 1;
            if constexpr (KIND == COB_VF) {
              if (GALE_IN_BOUNDS(M.err, pos >= fo[r] && pos < fo[r + 1])) GALE_ST(out_idx + base0 + pos, j);
            } else if (GALE_IN_BOUNDS(M.err, pos < Dm.fstar_cap) && pos < Dm.fstar_cap) {
              const int2 q = X.f_bc[j];
              fid[pos] = j;
              fp1[pos] = q.x == a ? q.y : -1;  // (x, a, y): y is above a; (x, y, a): no vertex above a
              fp2[pos] = -1;
            }
            ++pos;
          }
        }
      }
      for (int r = w; r < nrows; r += nw) {  // the own blocks
        const int o0 = ofirst[r], n_own = ofirst[r + 1] - o0, at = fo[r + 1] - n_own;
        for (int t = lane; t < n_own; t += 32) {
          if constexpr (KIND == COB_VF) {
            GALE_ST(out_idx + base0 + at + t, o0 + t);
          } else if (at + t < Dm.fstar_cap) {
            fid[at + t] = o0 + t;
            const int2 q = X.f_bc[o0 + t];
            fp1[at + t] = q.x;
            fp2[at + t] = q.y;
          }
        }
      }
    }
    if constexpr (KIND == COB_EF) __syncthreads();
  }
  // ---- C: one thread per row: members of the star, sizes -> offsets, write-out --------------------------
  if constexpr (ROWS) {
    for (int j = tid; j < n_tile_rows; j += NT) {
      const int r = rown[j];
      int st0, n;
      if constexpr (FROM_VT) { st0 = min(soff[r] - s_base, n_src); n = min(soff[r + 1] - s_base, n_src) - st0; }
      else { st0 = min(fo[r], Dm.fstar_cap); n = min(fo[r + 1], Dm.fstar_cap) - st0; }
      (void)GALE_IN_BOUNDS(M.err, n >= 0 && n <= 32 * W && r >= 0 && r < nrows);
      n = min(n, 32 * W);
      const int b = desc[KIND == COB_FT ? 2 * j : j];
      const int c = KIND == COB_FT ? desc[2 * j + 1] : 0;
      int cnt = 0;
      for (int k = 0; k < W; ++k) {
        uint32_t bits = 0u;
        const int e1 = min(32, n - 32 * k);
        for (int e = 0; e < e1; ++e) {
          bool hit;
          if constexpr (KIND == COB_EF) {
            hit = fp1[st0 + 32 * k + e] == b || fp2[st0 + 32 * k + e] == b;
          } else {
            const int at = st0 + 32 * k + e;         // a < b (< c): b is not the lowest vertex, c not one of the two lowest
            const int qy = ty[at], qz = tz[at], qw = tw[at];
            if constexpr (KIND == COB_ET) hit = qy == b || qz == b || qw == b;
            else hit = (qy == b || qz == b) && (qz == c || qw == c);
          }
          bits |= (uint32_t)hit << e;
        }
        rmask[j * W + k] = bits;
        cnt += __popc(bits);
      }
      rloc[j] = cnt;
    }
    __syncthreads();
    const int total = block_scan_smem(rloc, n_tile_rows, wsum);
    if (COUNT) {
      if (tid == 0) stats[tile] = total;
    } else {
      const int orow0 = P.row_base[slot] + (r_tile0 - first[v_lo - row_rel]);
      for (int j = tid; j < n_tile_rows; j += NT) {
        int off = base0 + rloc[j];
        out_off[orow0 + j] = off;
        const int r = rown[j];
        const int32_t* ids = KIND == COB_EF ? fid + min(fo[r], Dm.fstar_cap) : sid + min(soff[r] - s_base, n_src);
        for (int k = 0; k < W; ++k) {
          uint32_t bits = rmask[j * W + k];
          while (bits) {
            const int bpos = __ffs(bits) - 1;
            bits &= bits - 1;
            if (GALE_IN_BOUNDS(M.err, off < base0 + rloc[j + 1])) GALE_ST(out_idx + off, ids[k * 32 + bpos]);
            ++off;
          }
        }
      }
    }
  }
}

// ---- boundary relations FE / TE / TF by look-up --------------------------------------
// "Locate edge indices ... through the edge list E with limiting the search range by the edge interval array
// I_E": the edge (x, y), x < y, lies in the block [e_first[x], e_first[x+1]) of its lower vertex, which ascends
// with y; likewise a triangle (x, y, z) in the block of x of F, which ascends with (y, z). -1 = not in the list.
__device__ __forceinline__ int edge_id(const SubIndex& X, int x, int y) {
  int lo = __ldg(X.e_first + x), hi = __ldg(X.e_first + x + 1);
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(X.e_hi + mid) < y) lo = mid + 1; else hi = mid;
  }
  return (lo < __ldg(X.e_first + x + 1) && __ldg(X.e_hi + lo) == y) ? lo : -1;
}
__device__ __forceinline__ int triangle_id(const SubIndex& X, int x, int y, int z) {
  int lo = __ldg(X.f_first + x), hi = __ldg(X.f_first + x + 1);
  const int end = hi;
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    const int2 q = __ldg(X.f_bc + mid);
    if (q.x < y || (q.x == y && q.y < z)) lo = mid + 1; else hi = mid;
  }
  if (lo >= end) return -1;
  const int2 q = __ldg(X.f_bc + lo);
  return (q.x == y && q.y == z) ? lo : -1;
}

enum { BND_FE = 1, BND_TE = 2, BND_TF = 3 };
__host__ __device__ inline int boundary_width(int kind, int D) { return kind == BND_TF ? 4 : (kind == BND_FE ? 3 : (D == 4 ? 6 : 3)); }

// One thread per output entry: entry j of row r = the j-th vertex combination (lexicographic) of triangle
// first + r of F (FE) or of simplex first + r of T (TE, TF). out[r * width + j]; coalesced.
template <int KIND, int D>
__global__ void k_boundary(const SubIndex X, const int32_t* __restrict__ T, int nV, long long first, long long count, int32_t* out) {
  constexpr int W = KIND == BND_TF ? 4 : (KIND == BND_FE ? 3 : (D == 4 ? 6 : 3));
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= count * W) return;
  const long long r = e / W;
  const int j = (int)(e - r * W);
  const long long id = first + r;
  int v[4];
  if constexpr (KIND == BND_FE) {
    // (the three entries of a row repeat this search: the loads of the second and third hit the first's lines)
    // lowest vertex of triangle id: the vertex whose block of F holds it (last a with f_first[a] <= id)
    int lo = 0, hi = nV;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if ((long long)__ldg(X.f_first + mid) <= id) lo = mid; else hi = mid;
    }
    const int2 q = __ldg(X.f_bc + id);
    v[0] = lo; v[1] = q.x; v[2] = q.y; v[3] = 0;
  } else {
#pragma unroll
    for (int k = 0; k < D; ++k) v[k] = __ldg(T + id * D + k);
  }
  int res;
  if constexpr (KIND == BND_TF) {
    // (0,1,2) (0,1,3) (0,2,3) (1,2,3)
    const int a = j == 3 ? v[1] : v[0], b = j >= 2 ? v[2] : v[1], c = j == 0 ? v[2] : v[3];
    res = triangle_id(X, a, b, c);
  } else if (W == 3) {
    // (0,1) (0,2) (1,2)
    res = edge_id(X, j == 2 ? v[1] : v[0], j == 0 ? v[1] : v[2]);
  } else {
    // (0,1) (0,2) (0,3) (1,2) (1,3) (2,3)
    const int a = j < 3 ? v[0] : (j < 5 ? v[1] : v[2]);
    const int b = j == 0 ? v[1] : ((j == 1 || j == 3) ? v[2] : v[3]);
    res = edge_id(X, a, b);
  }
  out[e] = res;
}

}  // namespace sub
}  // namespace gale
