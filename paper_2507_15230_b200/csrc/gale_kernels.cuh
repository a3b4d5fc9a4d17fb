// gale_kernels.cuh — sm_100a kernels of the GALE relation hot path.
//
// One thread block owns one *tile*: a contiguous vertex sub-range [v_lo, v_hi) of a cluster
// (a tile plays the role of the paper's <=100-vertex segment; a cluster is the
// request unit). The block
//   a1  stages the tile's internal simplices (contiguous rows of T, I_T PAPER.md:178) and its
//       external ones (gathered through the tile's T_ex list) into shared memory,
//   a2  VT: counts incidences per local vertex with shared-memory atomics, scans, scatters, and
//       fixes the row order (rows are short); the simplices whose *lowest* vertex is v are the
//       contiguous run first_tet[v]..first_tet[v+1] and are written without atomics,
//   a3  VV: neighbours inside the tile go to a tile x tile bitmap (atomicOr), neighbours outside
//       it through a shared-memory open-addressing set of (row, vertex) keys ("no duplicates",
//       PAPER.md:228); rows come out ascending: [outside-below][bitmap][outside-above],
//   a4  TT: facets (sorted vertex tuples) are matched in a shared-memory open-addressing table;
//       an external simplex can only meet an internal one through its facet opposite its lowest
//       vertex, and only if its second vertex is in the tile, so it inserts at most one facet,
//   a5  TT fallback: the facet opposite the lowest vertex a of an internal simplex (a,b,..) whose
//       other vertices are all >= v_hi may have its coface outside the staged set; it is resolved
//       from global memory through the run of simplices starting with b and the index of
//       simplices whose second vertex is b (DESIGN.md §TT fallback),
//   a6  writes the CSR pieces with coalesced stores.
// All arithmetic is int32 index work; no floating point.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gale {

constexpr int kThreads = 256;          // threads per block; also the largest tile (rows per block)
constexpr int kMaxBatch = 128;         // clusters per kernel launch (descriptor lives in kernel params)
constexpr uint32_t kEmpty32 = 0xFFFFFFFFu;
constexpr unsigned long long kEmpty64 = ~0ull;
constexpr uint16_t kNoMate = 0xFFFFu;
constexpr int kMaxStaged = 16000;      // staged simplices per tile (16-bit record ids)

enum { REL_VT = 1, REL_VV = 2, REL_TT = 4 };
enum { ERR_VV_TABLE_FULL = 1, ERR_TT_TABLE_FULL = 2, ERR_SIZE_MISMATCH = 4, ERR_COUNT_ROW_TOO_BIG = 8 };

// Device-resident index built by gale_mesh_create (all pointers DEVICE).
struct DeviceMesh {
  const int32_t* T;                 // [nT*D] canonical simplices (caller's array)
  const int32_t* first_tet;         // [nV+1] first simplex whose lowest vertex is >= v  (I_T)
  const int32_t* opp_first;         // [nV+1] first position in opp_perm whose second vertex is >= v
  const int32_t* opp_perm;          // [nT]   simplex ids grouped by second vertex
  const int32_t* tile_vlo;          // [nTiles+1] tile i owns vertices [tile_vlo[i], tile_vlo[i+1])
  const long long* tex_off;         // [nTiles+1] offsets into tex
  const int32_t* tex;               // per-tile ascending ids of external simplices (T_ex)
  const long long* vt_pref;         // [nTiles+1] exclusive prefix of per-tile VT nnz
  const long long* vv_pref;         // [nTiles+1] exclusive prefix of per-tile VV nnz
  const int32_t* cluster_tile_begin;  // [nC+1]
  int32_t* err;                     // sticky device error flags
};

// Shared-memory capacities (maxima over all tiles of the mesh, fixed at create).
struct SmemCfg {
  int tv;        // rows (vertices) per tile
  int smax;      // staged simplices
  int sext;      // external simplices
  int sint;      // internal simplices
  int vt_max;    // VT entries
  int vv_max;    // VV entries
  int tth_cap;   // TT facet table slots (power of two)
  int vvh_cap;   // VV outside-pair table slots (power of two)
  int bm_words;  // bitmap words per row = ceil(tv/32)
};

struct SmemLayout {
  int tets, texid, ft, cnt_vt, cnt_lo, cnt_hi, pop, off_vt, off_vv, cur_vt, cur_lo, cur_hi, bm, vvh, tth, mate, vt_idx,
      vv_idx, scan, total;
};

__host__ __device__ inline int align16(int x) { return (x + 15) & ~15; }

__host__ __device__ inline SmemLayout make_layout(const SmemCfg& c, int D) {
  SmemLayout L;
  int o = 0;
  L.vvh = o;    o = align16(o + c.vvh_cap * 8);
  L.tets = o;   o = align16(o + c.smax * D * 4);
  L.texid = o;  o = align16(o + c.sext * 4);
  L.ft = o;     o = align16(o + (c.tv + 1) * 4);
  L.cnt_vt = o; o = align16(o + c.tv * 4);
  L.cnt_lo = o; o = align16(o + c.tv * 4);
  L.cnt_hi = o; o = align16(o + c.tv * 4);
  L.pop = o;    o = align16(o + c.tv * 4);
  L.off_vt = o; o = align16(o + (c.tv + 1) * 4);
  L.off_vv = o; o = align16(o + (c.tv + 1) * 4);
  L.cur_vt = o; o = align16(o + c.tv * 4);
  L.cur_lo = o; o = align16(o + c.tv * 4);
  L.cur_hi = o; o = align16(o + c.tv * 4);
  L.bm = o;     o = align16(o + c.tv * c.bm_words * 4);
  L.tth = o;    o = align16(o + c.tth_cap * 4);
  L.mate = o;   o = align16(o + c.sint * 4 * 2);
  L.vt_idx = o; o = align16(o + c.vt_max * 4);
  L.vv_idx = o; o = align16(o + c.vv_max * 4);
  L.scan = o;   o = align16(o + 80 * 4);
  L.total = o;
  return L;
}

// Per-launch batch descriptor, passed by value in kernel parameter space (no H2D copy).
struct BatchParams {
  int n_clusters;
  uint32_t mask;
  int total_rows;                    // VT/VV rows of the whole batch
  int total_vt_nnz, total_vv_nnz;    // terminal offsets
  int tile_prefix[kMaxBatch + 1];    // tiles of the batch before cluster slot i  (block -> cluster slot)
  int cluster[kMaxBatch];            // cluster id of slot i
  int row_base[kMaxBatch];           // first VT/VV row of slot i in the batch
  int vt_base[kMaxBatch];            // first VT index position of slot i
  int vv_base[kMaxBatch];
  int tt_base[kMaxBatch];            // first TT row of slot i
};

struct OutPtrs {
  int32_t* vt_offsets;
  int32_t* vt_indices;
  int32_t* vv_offsets;
  int32_t* vv_indices;
  int32_t* tt_indices;
};

// ------------------------------------------------------------------------------------------------
// Guard codes go to a host-mapped word (plain store: no PCIe atomics needed; any code is fatal).
__device__ __forceinline__ void raise_err(int32_t* err, int code) { *reinterpret_cast<volatile int32_t*>(err) = code; }

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async4(void* smem, const void* gmem) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

__device__ __forceinline__ uint32_t mix32(uint32_t h) {
  h ^= h >> 15;
  h *= 0x2C1B3C6Du;
  h ^= h >> 12;
  h *= 0x297A2D39u;
  h ^= h >> 15;
  return h;
}

template <int D>
__device__ __forceinline__ void load_simplex(const int32_t* tets, int i, int (&v)[D]) {
  if constexpr (D == 4) {
    const int4 q = reinterpret_cast<const int4*>(tets)[i];
    v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
  } else {
    v[0] = tets[i * 3]; v[1] = tets[i * 3 + 1]; v[2] = tets[i * 3 + 2];
  }
}
template <int D>
__device__ __forceinline__ void load_simplex_global(const int32_t* T, long long t, int (&v)[D]) {
  if constexpr (D == 4) {
    const int4 q = __ldg(reinterpret_cast<const int4*>(T) + t);
    v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
  } else {
    v[0] = __ldg(T + t * 3); v[1] = __ldg(T + t * 3 + 1); v[2] = __ldg(T + t * 3 + 2);
  }
}
// facet of v opposite its k-th vertex (ascending because v is)
template <int D>
__device__ __forceinline__ void facet_of(const int (&v)[D], int k, int (&f)[D - 1]) {
#pragma unroll
  for (int j = 0; j < D - 1; ++j) f[j] = (j < k) ? v[j] : v[j + 1];
}
template <int D>
__device__ __forceinline__ uint32_t facet_hash(const int (&f)[D - 1]) {
  uint32_t h = (uint32_t)f[0] * 0x9E3779B1u ^ (uint32_t)f[1] * 0x85EBCA77u;
  if constexpr (D == 4) h ^= (uint32_t)f[2] * 0xC2B2AE3Du;
  return mix32(h);
}

// Stage the tile's simplices: internal rows [t_lo, t_lo+s_int) then the external ones.
template <int D>
__device__ __forceinline__ void stage_tile(const DeviceMesh& M, int32_t* tets, int32_t* texid, int t_lo, int s_int,
                                           long long tex_b, int s_ext) {
  const int tid = threadIdx.x;
  if constexpr (D == 4) {
    const int4* src = reinterpret_cast<const int4*>(M.T) + t_lo;
    int4* dst = reinterpret_cast<int4*>(tets);
    for (int i = tid; i < s_int; i += kThreads) cp_async16(dst + i, src + i);
    for (int j = tid; j < s_ext; j += kThreads) {
      const int id = __ldg(M.tex + tex_b + j);
      texid[j] = id;
      cp_async16(dst + s_int + j, reinterpret_cast<const int4*>(M.T) + id);
    }
  } else {
    const int32_t* src = M.T + (long long)t_lo * 3;
    for (int i = tid; i < s_int * 3; i += kThreads) cp_async4(tets + i, src + i);
    for (int j = tid; j < s_ext; j += kThreads) {
      const int id = __ldg(M.tex + tex_b + j);
      texid[j] = id;
      const int32_t* g = M.T + (long long)id * 3;
      int32_t* d = tets + (s_int + j) * 3;
      cp_async4(d, g); cp_async4(d + 1, g + 1); cp_async4(d + 2, g + 2);
    }
  }
}

// Insert (row, outside vertex) into the VV set. Returns true if this call created the entry.
__device__ __forceinline__ bool vv_set_insert(unsigned long long* tbl, int cap, int row, int u, int32_t* err) {
  const unsigned long long key = ((unsigned long long)(uint32_t)row << 32) | (uint32_t)u;
  uint32_t slot = mix32((uint32_t)u * 0x9E3779B1u ^ (uint32_t)row * 0x85EBCA77u) & (cap - 1);
  for (int probe = 0; probe < cap; ++probe) {
    unsigned long long cur = tbl[slot];
    if (cur == key) return false;
    if (cur == kEmpty64) {
      cur = atomicCAS(&tbl[slot], kEmpty64, key);
      if (cur == kEmpty64) return true;
      if (cur == key) return false;
    }
    slot = (slot + 1) & (cap - 1);
  }
  raise_err(err, ERR_VV_TABLE_FULL);
  return false;
}

// Insert facet f of staged simplex i (record (i<<2)|k); on meeting its twin, join the two.
template <int D>
__device__ __forceinline__ void tt_insert(uint32_t* tbl, int cap, const int32_t* tets, uint16_t* mate, int s_int,
                                          const int (&f)[D - 1], int i, int k, int32_t* err) {
  const uint32_t h = facet_hash<D>(f);
  const uint32_t me = (h & 0xFFFF0000u) | (uint32_t)((i << 2) | k);
  uint32_t slot = h & (cap - 1);
  for (int probe = 0; probe < cap; ++probe) {
    uint32_t cur = tbl[slot];
    if (cur == kEmpty32) {
      cur = atomicCAS(&tbl[slot], kEmpty32, me);
      if (cur == kEmpty32) return;
    }
    if ((cur ^ me) < 0x10000u) {  // same fingerprint: compare the facets themselves
      const int oi = (cur & 0xFFFFu) >> 2, ok = cur & 3;
      int ov[D], of[D - 1];
      load_simplex<D>(tets, oi, ov);
      facet_of<D>(ov, ok, of);
      bool same = true;
#pragma unroll
      for (int j = 0; j < D - 1; ++j) same &= (of[j] == f[j]);
      if (same) {
        if (oi < s_int) mate[(oi << 2) | ok] = (uint16_t)i;
        if (i < s_int) mate[(i << 2) | k] = (uint16_t)oi;
        return;
      }
    }
    slot = (slot + 1) & (cap - 1);
  }
  raise_err(err, ERR_TT_TABLE_FULL);
}

// a5: coface of facet f (= simplex `self` minus its lowest vertex), looked up in global memory.
// Both cofaces of a facet with lowest vertex b have b as lowest or second-lowest vertex.
template <int D>
__device__ __noinline__ int tt_fallback(const DeviceMesh& M, const int (&f)[D - 1], int self) {
  const int b = f[0];
  // (i) simplices whose lowest vertex is b: contiguous run of T
  for (int s = __ldg(M.first_tet + b), e = __ldg(M.first_tet + b + 1); s < e; ++s) {
    int v[D];
    load_simplex_global<D>(M.T, s, v);
    int hit = 0;
#pragma unroll
    for (int j = 1; j < D - 1; ++j)
#pragma unroll
      for (int k = 1; k < D; ++k) hit += (v[k] == f[j]);
    if (hit == D - 2) return s;
  }
  // (ii) simplices whose second vertex is b: (y, b, f[1], ...)
  for (int p = __ldg(M.opp_first + b), e = __ldg(M.opp_first + b + 1); p < e; ++p) {
    const int s = __ldg(M.opp_perm + p);
    if (s == self) continue;
    int v[D];
    load_simplex_global<D>(M.T, s, v);
    bool same = true;
#pragma unroll
    for (int j = 1; j < D - 1; ++j) same &= (v[j + 1] == f[j]);
    if (same) return s;
  }
  return -1;
}

// Block-wide exclusive scan of one value per thread (kThreads threads). Returns the exclusive
// prefix; *total gets the block sum. scratch: 33 ints of shared memory.
__device__ __forceinline__ int block_exclusive_scan(int x, int* scratch, int* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int inc = x;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int y = __shfl_up_sync(0xFFFFFFFFu, inc, d);
    if (lane >= d) inc += y;
  }
  if (lane == 31) scratch[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int w = lane < (kThreads / 32) ? scratch[lane] : 0;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int y = __shfl_up_sync(0xFFFFFFFFu, w, d);
      if (lane >= d) w += y;
    }
    scratch[lane] = w;  // inclusive warp totals
  }
  __syncthreads();
  const int base = warp == 0 ? 0 : scratch[warp - 1];
  *total = scratch[kThreads / 32 - 1];
  const int r = base + inc - x;
  __syncthreads();
  return r;
}

__device__ __forceinline__ void insertion_sort(int32_t* a, int n) {
  for (int i = 1; i < n; ++i) {
    const int32_t x = a[i];
    int j = i - 1;
    while (j >= 0 && a[j] > x) {
      a[j + 1] = a[j];
      --j;
    }
    a[j + 1] = x;
  }
}

// ------------------------------------------------------------------------------------------------
// The batch kernel: VT + VV + TT for every tile of the requested clusters.
template <int D>
__global__ void __launch_bounds__(kThreads) gale_batch_kernel(const DeviceMesh M, const __grid_constant__ BatchParams P,
                                                              const SmemCfg C, const OutPtrs O) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x;
  const uint32_t mask = P.mask;

  if (blockIdx.x == 0 && tid == 0) {  // terminal offsets (also covers batches without rows)
    if (mask & REL_VT) { O.vt_offsets[0] = 0; O.vt_offsets[P.total_rows] = P.total_vt_nnz; }
    if (mask & REL_VV) { O.vv_offsets[0] = 0; O.vv_offsets[P.total_rows] = P.total_vv_nnz; }
  }
  if ((int)blockIdx.x >= P.tile_prefix[P.n_clusters]) return;

  // block -> (cluster slot, tile)
  int lo = 0, hi = P.n_clusters;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (P.tile_prefix[mid] <= (int)blockIdx.x) lo = mid; else hi = mid;
  }
  const int slot = lo;
  const int cl = P.cluster[slot];
  const int tile0 = __ldg(M.cluster_tile_begin + cl);
  const int tile = tile0 + ((int)blockIdx.x - P.tile_prefix[slot]);
  const int v_lo = __ldg(M.tile_vlo + tile), v_hi = __ldg(M.tile_vlo + tile + 1);
  const int nrows = v_hi - v_lo;
  const int cv_lo = __ldg(M.tile_vlo + tile0);                       // first vertex of the cluster
  const int t_lo = __ldg(M.first_tet + v_lo), t_hi = __ldg(M.first_tet + v_hi);
  const int ct_lo = __ldg(M.first_tet + cv_lo);                      // first internal simplex of the cluster
  const int s_int = t_hi - t_lo;
  const long long tex_b = __ldg(M.tex_off + tile);
  const int s_ext = (int)(__ldg(M.tex_off + tile + 1) - tex_b);
  const int S = s_int + s_ext;
  const int row0 = P.row_base[slot] + (v_lo - cv_lo);                // first output row of this tile
  const int vt0 = P.vt_base[slot] + (int)(__ldg(M.vt_pref + tile) - __ldg(M.vt_pref + tile0));
  const int vv0 = P.vv_base[slot] + (int)(__ldg(M.vv_pref + tile) - __ldg(M.vv_pref + tile0));
  const int tt0 = P.tt_base[slot] + (t_lo - ct_lo);                  // first TT row of this tile

  const SmemLayout L = make_layout(C, D);
  int32_t* tets = reinterpret_cast<int32_t*>(smem + L.tets);
  int32_t* texid = reinterpret_cast<int32_t*>(smem + L.texid);
  int32_t* ft = reinterpret_cast<int32_t*>(smem + L.ft);
  int32_t* cnt_vt = reinterpret_cast<int32_t*>(smem + L.cnt_vt);
  int32_t* cnt_lo = reinterpret_cast<int32_t*>(smem + L.cnt_lo);
  int32_t* cnt_hi = reinterpret_cast<int32_t*>(smem + L.cnt_hi);
  int32_t* popc = reinterpret_cast<int32_t*>(smem + L.pop);
  int32_t* off_vt = reinterpret_cast<int32_t*>(smem + L.off_vt);
  int32_t* off_vv = reinterpret_cast<int32_t*>(smem + L.off_vv);
  int32_t* cur_vt = reinterpret_cast<int32_t*>(smem + L.cur_vt);
  int32_t* cur_lo = reinterpret_cast<int32_t*>(smem + L.cur_lo);
  int32_t* cur_hi = reinterpret_cast<int32_t*>(smem + L.cur_hi);
  uint32_t* bm = reinterpret_cast<uint32_t*>(smem + L.bm);
  unsigned long long* vvh = reinterpret_cast<unsigned long long*>(smem + L.vvh);
  uint32_t* tth = reinterpret_cast<uint32_t*>(smem + L.tth);
  uint16_t* mate = reinterpret_cast<uint16_t*>(smem + L.mate);
  int32_t* vt_idx = reinterpret_cast<int32_t*>(smem + L.vt_idx);
  int32_t* vv_idx = reinterpret_cast<int32_t*>(smem + L.vv_idx);
  int* scan = reinterpret_cast<int*>(smem + L.scan);
  const int W = C.bm_words;

  // ---- a1: stage + clear ----------------------------------------------------------------------
  stage_tile<D>(M, tets, texid, t_lo, s_int, tex_b, s_ext);
  if (tid < nrows) {
    cnt_vt[tid] = 0; cnt_lo[tid] = 0; cnt_hi[tid] = 0; cur_vt[tid] = 0; cur_lo[tid] = 0; cur_hi[tid] = 0;
  }
  for (int i = tid; i <= nrows; i += kThreads) ft[i] = __ldg(M.first_tet + v_lo + i);
  if (mask & REL_VV) {
    for (int i = tid; i < nrows * W; i += kThreads) bm[i] = 0u;
    for (int i = tid; i < C.vvh_cap; i += kThreads) vvh[i] = kEmpty64;
  }
  if (mask & REL_TT) {
    for (int i = tid; i < C.tth_cap; i += kThreads) tth[i] = kEmpty32;
    uint32_t* m32 = reinterpret_cast<uint32_t*>(mate);
    for (int i = tid; i < s_int * 2; i += kThreads) m32[i] = 0xFFFFFFFFu;
  }
  cp_async_wait_all();
  __syncthreads();

  // ---- pass A: count VT, build the VV bitmap + outside set, match facets ----------------------
  for (int i = tid; i < S; i += kThreads) {
    int v[D];
    load_simplex<D>(tets, i, v);
    const bool is_int = i < s_int;
    bool in[D];
#pragma unroll
    for (int k = 0; k < D; ++k) in[k] = (unsigned)(v[k] - v_lo) < (unsigned)nrows;
#pragma unroll
    for (int k = 0; k < D; ++k) {
      if (!in[k]) continue;
      const int r = v[k] - v_lo;
      if ((mask & REL_VT) && k > 0) atomicAdd(&cnt_vt[r], 1);   // k == 0 <=> internal: counted by its run
      if (mask & REL_VV) {
#pragma unroll
        for (int j = 0; j < D; ++j) {
          if (j == k) continue;
          const int u = v[j];
          if (in[j]) {
            const int ul = u - v_lo;
            atomicOr(&bm[r * W + (ul >> 5)], 1u << (ul & 31));
          } else if (vv_set_insert(vvh, C.vvh_cap, r, u, M.err)) {
            atomicAdd(u < v_lo ? &cnt_lo[r] : &cnt_hi[r], 1);
          }
        }
      }
    }
    if (mask & REL_TT) {
      if (is_int) {
#pragma unroll
        for (int k = 0; k < D; ++k) {
          int f[D - 1];
          facet_of<D>(v, k, f);
          tt_insert<D>(tth, C.tth_cap, tets, mate, s_int, f, i, k, M.err);
        }
      } else if (in[1]) {
        int f[D - 1];
        facet_of<D>(v, 0, f);
        tt_insert<D>(tth, C.tth_cap, tets, mate, s_int, f, i, 0, M.err);
      }
    }
  }
  __syncthreads();

  // ---- row degrees -> offsets -----------------------------------------------------------------
  {
    int dvt = 0, dvv = 0;
    if (tid < nrows) {
      dvt = cnt_vt[tid] + (ft[tid + 1] - ft[tid]);
      if (mask & REL_VV) {
        int p = 0;
        for (int w = 0; w < W; ++w) p += __popc(bm[tid * W + w]);
        popc[tid] = p;
        dvv = cnt_lo[tid] + p + cnt_hi[tid];
      }
    }
    int tot_vt, tot_vv = 0;
    const int evt = block_exclusive_scan(dvt, scan, &tot_vt);
    if (tid < nrows) off_vt[tid] = evt;
    if (tid == 0) off_vt[nrows] = tot_vt;
    if (mask & REL_VV) {
      const int evv = block_exclusive_scan(dvv, scan + 33, &tot_vv);
      if (tid < nrows) off_vv[tid] = evv;
      if (tid == 0) off_vv[nrows] = tot_vv;
    }
    if (tid == 0) {  // the sizes fixed at create must be reproduced exactly
      const int evt_n = (int)(__ldg(M.vt_pref + tile + 1) - __ldg(M.vt_pref + tile));
      const int evv_n = (int)(__ldg(M.vv_pref + tile + 1) - __ldg(M.vv_pref + tile));
      if (((mask & REL_VT) && tot_vt != evt_n) || ((mask & REL_VV) && tot_vv != evv_n)) raise_err(M.err, ERR_SIZE_MISMATCH);
    }
    if (tid < nrows) {
      if (mask & REL_VT) O.vt_offsets[row0 + tid] = vt0 + evt;
      if (mask & REL_VV) O.vv_offsets[row0 + tid] = vv0 + off_vv[tid];
    }
    if (tid == 0) {
      if (mask & REL_VT) O.vt_offsets[row0 + nrows] = vt0 + tot_vt;
      if (mask & REL_VV) O.vv_offsets[row0 + nrows] = vv0 + tot_vv;
    }
  }
  __syncthreads();

  // ---- pass B: scatter VT, read back TT, place the outside VV entries -------------------------
  for (int i = tid; i < S; i += kThreads) {
    int v[D];
    load_simplex<D>(tets, i, v);
    const bool is_int = i < s_int;
    const int gid = is_int ? t_lo + i : texid[i - s_int];
    if (mask & REL_VT) {
#pragma unroll
      for (int k = 1; k < D; ++k) {
        const int r = v[k] - v_lo;
        if ((unsigned)r < (unsigned)nrows) vt_idx[off_vt[r] + atomicAdd(&cur_vt[r], 1)] = gid;
      }
      if (is_int) {
        const int r = v[0] - v_lo;
        vt_idx[off_vt[r] + cnt_vt[r] + (gid - ft[r])] = gid;
      }
    }
    if ((mask & REL_TT) && is_int) {
      int nb[D];
#pragma unroll
      for (int k = 0; k < D; ++k) {
        const uint16_t m = mate[(i << 2) | k];
        if (m != kNoMate) {
          nb[k] = (int)m < s_int ? t_lo + (int)m : texid[(int)m - s_int];
        } else if (k == 0 && v[1] >= v_hi) {
          int f[D - 1];
          facet_of<D>(v, 0, f);
          nb[k] = tt_fallback<D>(M, f, gid);
        } else {
          nb[k] = -1;
        }
      }
      if constexpr (D == 4) {
        reinterpret_cast<int4*>(O.tt_indices)[tt0 + i] = make_int4(nb[0], nb[1], nb[2], nb[3]);
      } else {
        int32_t* o = O.tt_indices + (long long)(tt0 + i) * 3;
        o[0] = nb[0]; o[1] = nb[1]; o[2] = nb[2];
      }
    }
  }
  if (mask & REL_VV) {
    for (int s = tid; s < C.vvh_cap; s += kThreads) {
      const unsigned long long key = vvh[s];
      if (key == kEmpty64) continue;
      const int r = (int)(key >> 32), u = (int)(uint32_t)key;
      const int pos = u < v_lo ? off_vv[r] + atomicAdd(&cur_lo[r], 1)
                               : off_vv[r] + cnt_lo[r] + popc[r] + atomicAdd(&cur_hi[r], 1);
      vv_idx[pos] = u;
    }
  }
  __syncthreads();

  // ---- per row: order the atomically-placed parts, expand the bitmap --------------------------
  if (tid < nrows) {
    if (mask & REL_VT) insertion_sort(vt_idx + off_vt[tid], cnt_vt[tid]);
    if (mask & REL_VV) {
      int32_t* row = vv_idx + off_vv[tid];
      insertion_sort(row, cnt_lo[tid]);
      int p = cnt_lo[tid];
      for (int w = 0; w < W; ++w) {
        uint32_t bits = bm[tid * W + w];
        while (bits) {
          const int b = __ffs(bits) - 1;
          bits &= bits - 1;
          row[p++] = v_lo + w * 32 + b;
        }
      }
      insertion_sort(row + p, cnt_hi[tid]);
    }
  }
  __syncthreads();

  // ---- a6: coalesced write-out ----------------------------------------------------------------
  if (mask & REL_VT) {
    const int n = off_vt[nrows];
    for (int i = tid; i < n; i += kThreads) O.vt_indices[vt0 + i] = vt_idx[i];
  }
  if (mask & REL_VV) {
    const int n = off_vv[nrows];
    for (int i = tid; i < n; i += kThreads) O.vv_indices[vv0 + i] = vv_idx[i];
  }
}

// ------------------------------------------------------------------------------------------------
// Create-time sizing kernel: per tile, the exact VT and VV entry counts, the number of distinct
// outside (row, vertex) pairs and the number of facet records (a count-only run of a2-a4; the
// paper's leader producer likewise sizes its relation arrays before launch).
// The outside-pair set is processed in row chunks so a fixed-size table can never overflow.
struct CountCfg {
  int tv, smax, sext, hcap, bm_words;
};
struct CountLayout {
  int tets, texid, deg, bm, hash, misc, total;
};
__host__ __device__ inline CountLayout make_count_layout(const CountCfg& c, int D) {
  CountLayout L;
  int o = 0;
  L.hash = o;  o = align16(o + c.hcap * 8);
  L.tets = o;  o = align16(o + c.smax * D * 4);
  L.texid = o; o = align16(o + c.sext * 4);
  L.deg = o;   o = align16(o + c.tv * 4);
  L.bm = o;    o = align16(o + c.tv * c.bm_words * 4);
  L.misc = o;  o = align16(o + 16 * 4);
  L.total = o;
  return L;
}

template <int D>
__global__ void __launch_bounds__(kThreads) gale_count_kernel(const DeviceMesh M, const CountCfg C, int num_tiles,
                                                              long long* stats /*[num_tiles][4]*/) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x;
  const int tile = blockIdx.x;
  if (tile >= num_tiles) return;
  const CountLayout L = make_count_layout(C, D);
  int32_t* tets = reinterpret_cast<int32_t*>(smem + L.tets);
  int32_t* texid = reinterpret_cast<int32_t*>(smem + L.texid);
  int32_t* deg = reinterpret_cast<int32_t*>(smem + L.deg);
  uint32_t* bm = reinterpret_cast<uint32_t*>(smem + L.bm);
  unsigned long long* hash = reinterpret_cast<unsigned long long*>(smem + L.hash);
  int* misc = reinterpret_cast<int*>(smem + L.misc);  // [0] unique outside, [1] tt records, [2] chunk lo, [3] chunk hi
  const int W = C.bm_words;

  const int v_lo = __ldg(M.tile_vlo + tile), v_hi = __ldg(M.tile_vlo + tile + 1);
  const int nrows = v_hi - v_lo;
  const int t_lo = __ldg(M.first_tet + v_lo), t_hi = __ldg(M.first_tet + v_hi);
  const int s_int = t_hi - t_lo;
  const long long tex_b = __ldg(M.tex_off + tile);
  const int s_ext = (int)(__ldg(M.tex_off + tile + 1) - tex_b);
  const int S = s_int + s_ext;

  stage_tile<D>(M, tets, texid, t_lo, s_int, tex_b, s_ext);
  if (tid < nrows) deg[tid] = 0;
  for (int i = tid; i < nrows * W; i += kThreads) bm[i] = 0u;
  if (tid < 4) misc[tid] = 0;
  cp_async_wait_all();
  __syncthreads();

  for (int i = tid; i < S; i += kThreads) {
    int v[D];
    load_simplex<D>(tets, i, v);
    bool in[D];
#pragma unroll
    for (int k = 0; k < D; ++k) in[k] = (unsigned)(v[k] - v_lo) < (unsigned)nrows;
#pragma unroll
    for (int k = 0; k < D; ++k) {
      if (!in[k]) continue;
      const int r = v[k] - v_lo;
      atomicAdd(&deg[r], 1);
#pragma unroll
      for (int j = 0; j < D; ++j)
        if (j != k && in[j]) {
          const int ul = v[j] - v_lo;
          atomicOr(&bm[r * W + (ul >> 5)], 1u << (ul & 31));
        }
    }
    if (i < s_int) atomicAdd(&misc[1], D);
    else if (in[1]) atomicAdd(&misc[1], 1);
  }
  __syncthreads();

  // outside pairs, in row chunks whose candidate count fits the table at load <= 1/2
  int row_lo = 0;
  while (row_lo < nrows) {
    if (tid == 0) {
      int r = row_lo, cand = 0;
      while (r < nrows && (cand + (D - 1) * deg[r]) * 2 <= C.hcap) { cand += (D - 1) * deg[r]; ++r; }
      if (r == row_lo) { raise_err(M.err, ERR_COUNT_ROW_TOO_BIG); r = row_lo + 1; }
      misc[2] = row_lo; misc[3] = r;
    }
    for (int i = tid; i < C.hcap; i += kThreads) hash[i] = kEmpty64;
    __syncthreads();
    const int c_lo = misc[2], c_hi = misc[3];
    for (int i = tid; i < S; i += kThreads) {
      int v[D];
      load_simplex<D>(tets, i, v);
#pragma unroll
      for (int k = 0; k < D; ++k) {
        const int r = v[k] - v_lo;
        if (r < c_lo || r >= c_hi) continue;
#pragma unroll
        for (int j = 0; j < D; ++j) {
          if (j == k) continue;
          if ((unsigned)(v[j] - v_lo) < (unsigned)nrows) continue;
          if (vv_set_insert(hash, C.hcap, r, v[j], M.err)) atomicAdd(&misc[0], 1);
        }
      }
    }
    __syncthreads();
    row_lo = c_hi;
  }

  // totals
  int dvt = 0, dvv = 0;
  if (tid < nrows) {
    dvt = deg[tid];
    for (int w = 0; w < W; ++w) dvv += __popc(bm[tid * W + w]);
  }
  __shared__ int red[66];
  int tvt, tvv;
  block_exclusive_scan(dvt, red, &tvt);
  block_exclusive_scan(dvv, red + 33, &tvv);
  if (tid == 0) {
    stats[tile * 4 + 0] = tvt;
    stats[tile * 4 + 1] = tvv + misc[0];
    stats[tile * 4 + 2] = misc[0];
    stats[tile * 4 + 3] = misc[1];
  }
}

}  // namespace gale
