// gale_kernels.cuh — sm_100a kernels of the GALE relation hot path.
//
// One thread block owns one *tile*: a contiguous vertex sub-range [v_lo, v_lo+nrows) of a cluster
// (a tile plays the role of the paper's <=100-vertex segment; a cluster is the
// request unit). gale_mesh_create stores, per tile, the simplices incident to it
// (internal ones = rows I_T of T; external ones = the tile's T_ex list)
// re-encoded in *tile-local* vertex ids (8-bit when no tile of the mesh has more than 255 local
// vertices, template argument LB = 1, else 16-bit) that ascend with the global id:
//     [lower halo 0..nlo) [tile vertices nlo..nlo+nrows) [upper halo ..nloc)
// ("halo" = vertices outside the tile that share a simplex with it), external simplices first.
// Every external simplex has a smaller global id than every internal one (its lowest vertex lies
// below the tile), so the staged order s = 0..S-1 ascends with the global simplex id.
//
// A block has NT = 2 * TV threads: two threads per tile vertex p, an "A" thread (tid = p) and a
// "B" thread (tid = TV + p), so that lanes of a warp are consecutive vertices (their bitmap rows
// and tables fall into distinct shared-memory banks). Phases:
//   P0  stage the list (4*LB bytes per simplex), the external simplices' global ids, the
//       local->global vertex table gid and, parallel to it, hft = (first_tet[g], first_tet[g+1]) of
//       every local vertex (the interval array I_T, restricted to the tile and its
//       halo) into shared memory with 16-byte cp.async; clear the bitmaps and tables;
//   P1  VT incidence bits, one thread per staged simplex: bit (row v, column s) for every tile
//       vertex v of s other than its lowest vertex (the simplices whose *lowest* vertex is v are
//       the contiguous run hft[v], and need no bits); for an internal simplex whose
//       second vertex b lies outside the tile, an L2 prefetch of the rows of T that P5 will read;
//   P2  row degrees (popc) -> exclusive scan -> VT offsets;
//   P3  A(p): walks the set bits of row p in ascending order = VT(p) without its run, already
//             sorted; per simplex: emit the VT entry, OR the simplex's vertices into VV row p
//             (the thread owns the row: "no duplicates", without contention), and
//             flag the entry when p is the simplex's second vertex;
//       B(p): walks the run of p: VT entries, VV bits, and the TT facet records 1..D-1 of every
//             simplex of the run into p's private open-addressing table;
//   P4  A(p): the flagged entries are the simplices (x, p, ..): their facet 0 has lowest vertex p
//             and joins p's table. A facet whose lowest vertex is p has all its cofaces among
//             run(p) and those simplices, so the second arrival of a key meets the first and both
//             TT entries are written (no atomics, no global traffic);
//       B(p): VV row p -> degree -> scan -> expansion (sorted because local ids ascend);
//   P5  TT rows, VT and VV indices are translated to global ids and written with coalesced
//       stores; the facet opposite the lowest vertex a of an internal simplex (a, b, ..) with b
//       outside the tile belongs to no vertex of the tile: such facets are queued and resolved
//       one per thread from global memory: first the run of simplices starting with b (its bounds
//       come from hft: one round trip; measured > 99 % of the cofaces are found there), else the
//       index of simplices whose second vertex is b.
// All arithmetic is integer index work; no floating point.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gale {

constexpr int kMaxBatch = 128;         // clusters per kernel launch (descriptor lives in kernel params)
constexpr uint32_t kEmpty32 = 0xFFFFFFFFu;
constexpr int kMaxStaged4 = 4094;      // tetrahedra: 12-bit staged index in a table word
constexpr int kMaxStaged3 = 16382;     // triangles: 14-bit staged index
constexpr int kMaxLocal4 = 512;        // tetrahedra: 9-bit local ids (18-bit facet key)
constexpr int kMaxLocal3 = 65534;      // triangles: 16-bit local ids
constexpr int kMaxNnz16 = 65535;       // VT / VV entries of one tile (16-bit packed scans)
constexpr int kMaxTileVertices = 256;

enum { REL_VT = 1, REL_VV = 2, REL_TT = 4, MODE_COUNT = 8 };
enum { ERR_TT_TABLE_FULL = 2, ERR_SIZE_MISMATCH = 4, ERR_BOUNDS = 8 };

// Per-tile record built by gale_mesh_create (80 bytes, 16-byte aligned).
struct TileDesc {
  int32_t v_lo, nrows;        // vertices [v_lo, v_lo+nrows)
  int32_t t_lo, s_int;        // internal simplices [t_lo, t_lo+s_int)
  int32_t s_ext;              // external simplices (T_ex of the tile)
  int32_t nlo, nloc;          // halo vertices below v_lo / local ids in total (halo + rows)
  int32_t row_rel, tt_rel;    // first row / first TT row of the tile inside its cluster
  int32_t vt_rel, vv_rel;     // first VT / VV entry of the tile inside its cluster
  int32_t vt_nnz, vv_nnz;     // entries of the tile (fixed at create; the kernel re-derives them)
  int32_t pad0;
  long long stg_off;          // first staged simplex of the tile in DeviceMesh::loc (multiple of 4)
  long long tex_off;          // first entry in DeviceMesh::tex (multiple of 4)
  long long gid_off;          // first entry in DeviceMesh::gid (multiple of 4)
};
static_assert(sizeof(TileDesc) == 80, "TileDesc layout");

// Device-resident index built by gale_mesh_create (all pointers DEVICE).
struct DeviceMesh {
  const int32_t* T;                   // [nT*D] canonical simplices (caller's array)
  const int32_t* first_tet;           // [nV+1] first simplex whose lowest vertex is >= v  (I_T)
  const int32_t* opp_first;           // [nV+1] first position in opp_perm whose second vertex is >= v
  const int32_t* opp_perm;            // [nT]   simplex ids grouped by second vertex
  const TileDesc* tiles;              // [nTiles]
  const void* loc;                    // staged simplices in tile-local ids: 4 x uint16 each, or 4 x uint8
                                      //   when no tile of the mesh has more than 255 local vertices (SmemCfg::lb)
  const int32_t* tex;                 // per-tile ascending global ids of external simplices (T_ex)
  const int32_t* gid;                 // per-tile global vertex id of every local id (ascending)
  const int2* hft;                    // per-tile, parallel to gid: (first_tet[g], first_tet[g+1]) — the
                                      //   interval array I_T restricted to the tile's vertices + halo
  const int32_t* cluster_tile_begin;  // [nC+1]
  int32_t* err;                       // sticky device error flags (host-mapped)
};

// Shared-memory capacities (maxima over all tiles of the mesh, fixed at create). A field is 0 when
// the launch's relation mask does not need the region.
struct SmemCfg {
  int tv;        // rows (vertices) per tile, <= NT/2
  int smax;      // staged simplices (multiple of 4)
  int lb;        // bytes per local vertex id in the staged list: 1 or 2
  int sext;      // external simplices (multiple of 4)
  int nloc;      // local vertex ids (multiple of 4)
  int sint;      // internal simplices (even): TT rows + fallback queue, 0 without TT
  int hs;        // table slots per tile vertex (even, so that the row stride hs+1 is odd), 0 without TT
  int WT;        // VT bitmap words per row (odd)
  int WV;        // VV bitmap words per row (odd), 0 without VV
  int vt_max;    // VT entries staged for write-out (16-bit)
  int vv_max;    // VV entries staged for write-out (16-bit), 0 without VV or in count mode
};

// Byte offsets of the shared-memory regions, computed on the host (make_layout) and passed as a
// kernel parameter.
struct SmemLayout {
  int tets, texid, gid, hft, off_vt, off_vv, cnt, fbq, scan, bmT, bmV, bm_end;
  int tbl, ttrow, tt_end;
  int st_vt, st_vv;
  int total;
};

__host__ __device__ inline int align16(int x) { return (x + 15) & ~15; }

template <int D>
__host__ __device__ inline SmemLayout make_layout(const SmemCfg& c) {
  SmemLayout L;
  int o = 0;
  L.tets = o;   o = align16(o + c.smax * 4 * c.lb);
  L.texid = o;  o = align16(o + c.sext * 4);
  L.gid = o;    o = align16(o + c.nloc * 4);
  L.hft = o;    o = align16(o + c.nloc * 8);
  L.off_vt = o; o = align16(o + (c.tv + 1) * 4);
  L.off_vv = o; o = align16(o + (c.tv + 1) * 4);
  L.cnt = o;    o = align16(o + c.tv * 4);
  L.scan = o;   o = align16(o + 48 * 4);
  // VT bitmap (P1-P3); afterwards the same bytes hold the VV staging area (written in P4) and the
  // fallback queue (written in P5)
  L.bmT = o;
  {
    const int bm = align16(c.tv * c.WT * 4);
    L.st_vv = o;
    L.fbq = o + align16(c.vv_max * 2);
    const int reuse = align16(c.vv_max * 2) + align16(c.sint * 2);
    o += bm > reuse ? bm : reuse;
  }
  L.bmV = o;    o = align16(o + c.tv * c.WV * 4);
  L.bm_end = o;
  L.tbl = o;    o = align16(o + (c.hs ? c.tv * (c.hs + 1) * 4 : 0));
  L.ttrow = o;  o = align16(o + c.sint * D * 2);
  L.tt_end = o;
  L.st_vt = o;  o = align16(o + c.vt_max * 2);
  L.total = o;
  return L;
}

// Per-launch batch descriptor, passed by value in kernel parameter space (no H2D copy).
struct BatchParams {
  int n_clusters;
  uint32_t mask;
  int tile_base;                     // count mode: first tile of the launch
  int total_rows;                    // VT/VV rows of the whole batch
  int total_vt_nnz, total_vv_nnz;    // terminal offsets
  int uniform_tiles;                 // > 0: every cluster of the batch has this many tiles (slot = block / it)
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
  long long* stats;                  // count mode: [nTiles][4] = VT nnz, VV nnz, 0, 0
};

// Bounds-checked build (-DGALE_CHECK_BOUNDS=1, libgale_checked.so; tests/test_gpu_bounds.py): every tile
// is checked against the launch's shared-memory capacities and every computed staging index before it
// is written; a violation raises ERR_BOUNDS through the device error word and skips the write.
// compute-sanitizer is not available on the build pool, this is its stand-in. Off by default: no code.
__device__ __forceinline__ void raise_err(int32_t* err, int code);
// Output stores: the CSR arrays are written once and never read by the kernels, so the stores are marked
// evict-first (st.global.cs) and leave L2 to the data the fall-back look-ups re-read. Measured +0.7 %
// (24.18 / 24.19 vs 24.36 / 24.36 G tets/s, alternating runs); -DGALE_STREAM_OUT=0 restores plain stores.
#ifndef GALE_STREAM_OUT
#define GALE_STREAM_OUT 1
#endif
#if GALE_STREAM_OUT
#define GALE_ST(ptr, val) __stcs((ptr), (val))
#else
#define GALE_ST(ptr, val) (*(ptr) = (val))
#endif

#ifndef GALE_CHECK_BOUNDS
#define GALE_CHECK_BOUNDS 0
#endif
#if GALE_CHECK_BOUNDS
#define GALE_IN_BOUNDS(err, cond) ((cond) ? true : (raise_err((err), ERR_BOUNDS), false))
#else
#define GALE_IN_BOUNDS(err, cond) true
#endif

// ------------------------------------------------------------------------------------------------
// Guard codes go to a host-mapped word (plain store: no PCIe atomics needed; any code is fatal).
__device__ __forceinline__ void raise_err(int32_t* err, int code) { *reinterpret_cast<volatile int32_t*>(err) = code; }

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

// Barrier among the `count` threads that name the same id (ids 1..15; 0 is __syncthreads).
__device__ __forceinline__ void named_barrier(int id, int count) {
  asm volatile("bar.sync %0, %1;\n" ::"r"(id), "r"(count) : "memory");
}

// Local vertex ids of staged simplex s (LB bytes each).
template <int LB>
__device__ __forceinline__ void load_local(const unsigned char* tets, int s, int (&l)[4]) {
  if constexpr (LB == 2) {
    const uint2 q = reinterpret_cast<const uint2*>(tets)[s];
    l[0] = q.x & 0xFFFF; l[1] = q.x >> 16; l[2] = q.y & 0xFFFF; l[3] = q.y >> 16;
  } else {
    const uint32_t q = reinterpret_cast<const uint32_t*>(tets)[s];
    l[0] = q & 0xFF; l[1] = (q >> 8) & 0xFF; l[2] = (q >> 16) & 0xFF; l[3] = q >> 24;
  }
}

// 1 << (l mod 32)
__device__ __forceinline__ uint32_t bit_of(int l) { return 1u << (l & 31); }

// a5, one request per thread: coface != self of the facet (b, c[, d]) (ascending global ids) whose
// vertices all lie outside the tile. [f0, f1) = run of simplices starting with b (from the tile's hft). Both cofaces of a facet with lowest vertex b have b as
// lowest or second-lowest vertex: candidates are the run of simplices starting with b and the
// simplices whose second vertex is b (those are (x, b, c, d) exactly). Candidates are fetched four
// at a time without early exit so that their loads overlap.
template <int D>
__device__ __forceinline__ int tt_fallback(const DeviceMesh& M, int f0, int f1, int b, int c, int d, int self) {
  int found = -1;
  if constexpr (D == 4) {
    const int4* T4 = reinterpret_cast<const int4*>(M.T);
    for (int t = f0; t < f1; t += 4) {
      int4 q[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) q[u] = __ldg(T4 + min(t + u, f1 - 1));
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const bool hit = (q[u].y == c && (q[u].z == d || q[u].w == d)) || (q[u].z == c && q[u].w == d);
        if (hit) found = min(t + u, f1 - 1);
      }
    }
    if (found >= 0) return found;  // measured: > 99 % of the cofaces start with b
    const int o0 = __ldg(M.opp_first + b), o1 = __ldg(M.opp_first + b + 1);
    for (int j = o0; j < o1; j += 4) {
      int t[4];
      int4 q[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) t[u] = __ldg(M.opp_perm + min(j + u, o1 - 1));
#pragma unroll
      for (int u = 0; u < 4; ++u) q[u] = __ldg(T4 + t[u]);
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (t[u] != self && q[u].z == c && q[u].w == d) found = t[u];
    }
  } else {
    for (int t = f0; t < f1; ++t) {
      const int v1 = __ldg(M.T + (long long)t * 3 + 1), v2 = __ldg(M.T + (long long)t * 3 + 2);
      if (v1 == c || v2 == c) found = t;
    }
    if (found >= 0) return found;
    const int o0 = __ldg(M.opp_first + b), o1 = __ldg(M.opp_first + b + 1);
    for (int j = o0; j < o1; ++j) {
      const int t = __ldg(M.opp_perm + j);
      if (t != self && __ldg(M.T + (long long)t * 3 + 2) == c) found = t;
    }
  }
  return found;
}

// Block-wide exclusive scan of one value per thread. Returns the exclusive prefix; *total gets
// the block sum. scratch: 33 ints of shared memory. Ends with all threads past the last barrier.
template <int NT>
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t x, uint32_t* scratch, uint32_t* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t inc = x;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, inc, d);
    if (lane >= d) inc += y;
  }
  if (lane == 31) scratch[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    uint32_t w = lane < (NT / 32) ? scratch[lane] : 0u;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, w, d);
      if (lane >= d) w += y;
    }
    scratch[lane] = w;  // inclusive warp totals
  }
  __syncthreads();
  const uint32_t base = warp == 0 ? 0u : scratch[warp - 1];
  *total = scratch[NT / 32 - 1];
  return base + inc - x;
}

// ------------------------------------------------------------------------------------------------
// TT tables. A table word of vertex p's group = key | s << kKeyBits | k << 30: the facet's
// vertices other than p (local ids, ascending), the staged simplex s it belongs to, and the local
// vertex k it is opposite to.
template <int D>
struct FacetBits {
  static constexpr int kKeyBits = D == 4 ? 18 : 16;
  static constexpr uint32_t kKeyMask = (1u << kKeyBits) - 1u;
  static constexpr uint32_t kIdxMask = (1u << (30 - kKeyBits)) - 1u;
};

struct GroupCtx {
  uint32_t* tbl;       // this vertex's table, hs slots
  uint32_t hs;         // slots (any size >= the group's records: a group never overflows its table)
  uint16_t* ttrow;     // TT rows of the tile's internal simplices as staged indices, 0xFFFF = none
  int s_ext;
  int s_all;           // staged simplices of the tile (bounds-checked build)
};

// Place facet k of staged simplex s with key `key`: claim an empty slot, or meet the record that
// holds the same key (the other coface) and write both TT entries.
template <int D>
__device__ __forceinline__ void group_place(const GroupCtx& g, uint32_t key, int s, int k, int32_t* err) {
  using FB = FacetBits<D>;
  uint32_t h = __umulhi(key * 0x9E3779B1u, g.hs);
  uint32_t cur = g.tbl[h];
  uint32_t probe = 0;
  while (cur != kEmpty32 && (cur & FB::kKeyMask) != key) {  // probe loop kept minimal: lanes diverge here
    h = h + 1 == g.hs ? 0u : h + 1;
    cur = g.tbl[h];
    if (++probe >= g.hs) { raise_err(err, ERR_TT_TABLE_FULL); return; }
  }
  if (!GALE_IN_BOUNDS(err, h < g.hs && (uint32_t)s <= FB::kIdxMask && key <= FB::kKeyMask && k >= 0 && k < D)) return;
  if (cur == kEmpty32) {
    g.tbl[h] = key | ((uint32_t)s << FB::kKeyBits) | ((uint32_t)k << 30);
  } else {
    const int s2 = (int)((cur >> FB::kKeyBits) & FB::kIdxMask), k2 = (int)(cur >> 30);
    if (!GALE_IN_BOUNDS(err, s < g.s_all && s2 < g.s_all && k2 < D)) return;
    if (s >= g.s_ext) g.ttrow[(s - g.s_ext) * D + k] = (uint16_t)s2;
    if (s2 >= g.s_ext) g.ttrow[(s2 - g.s_ext) * D + k2] = (uint16_t)s;
  }
}

// Key of the facet opposite local vertex K: the facet's vertices other than its lowest one.
template <int D, int K>
__device__ __forceinline__ uint32_t group_key(const int (&l)[4]) {
  if constexpr (D == 4) {
    const int a = K <= 1 ? l[2] : l[1];
    const int b = K == 3 ? l[2] : l[3];
    return (uint32_t)a | ((uint32_t)b << 9);
  } else {
    return (uint32_t)(K <= 1 ? l[2] : l[1]);
  }
}

// Exclusive scan over the B half of the block (threads [NT/2, NT)), one value per thread, with a
// named barrier so that the A half is not held up. Returns the exclusive prefix; *total = sum.
template <int NT>
__device__ __forceinline__ uint32_t half_exclusive_scan(uint32_t x, uint32_t* scratch, uint32_t* total) {
  constexpr int TV = NT / 2;
  const int lane = threadIdx.x & 31, warp = (threadIdx.x - TV) >> 5;
  uint32_t inc = x;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, inc, d);
    if (lane >= d) inc += y;
  }
  if constexpr (TV <= 32) {
    *total = __shfl_sync(0xFFFFFFFFu, inc, 31);
    return inc - x;
  } else {
    constexpr int NW = TV / 32;
    if (lane == 31) scratch[warp] = inc;
    named_barrier(1, TV);
    uint32_t base = 0u, tot = 0u;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      const uint32_t v = scratch[w];
      if (w < warp) base += v;
      tot += v;
    }
    named_barrier(1, TV);  // scratch may be reused
    *total = tot;
    return base + inc - x;
  }
}

// ------------------------------------------------------------------------------------------------
// The batch kernel: VT + VV + TT for every tile of the requested clusters (or, COUNT, the exact
// VT / VV sizes of tiles [tile_base, tile_base + gridDim.x) — the paper's leader producer likewise
// sizes its relation arrays before launch). NT = 2 * (rows per tile capacity).
template <int D, int NT, bool COUNT, int LB>
__global__ void __launch_bounds__(NT, (NT <= 64 ? 16 : (NT <= 128 ? 8 : (NT <= 256 ? 4 : 2))))
gale_batch_kernel(const DeviceMesh M, const __grid_constant__ BatchParams P, const SmemCfg C,
                  const SmemLayout L, const OutPtrs O) {
  extern __shared__ __align__(16) unsigned char smem[];
  constexpr int TV = NT / 2;
  const int tid = threadIdx.x, lane = tid & 31;
  const uint32_t mask = P.mask;
  const bool do_vt = (mask & REL_VT) != 0, do_vv = (mask & REL_VV) != 0;
  const bool do_tt = !COUNT && (mask & REL_TT) != 0;
  const bool entries = !COUNT && (do_vt || do_tt);  // VT entries are staged (TT reads their flags)

  // ---- block -> (cluster slot, tile) ----------------------------------------------------------
  int slot = 0, tile;
  if (COUNT) {
    tile = P.tile_base + (int)blockIdx.x;
  } else {
    if (blockIdx.x == 0 && tid == 0) {  // terminal offsets (also covers batches without rows)
      if (do_vt) { O.vt_offsets[0] = 0; O.vt_offsets[P.total_rows] = P.total_vt_nnz; }
      if (do_vv) { O.vv_offsets[0] = 0; O.vv_offsets[P.total_rows] = P.total_vv_nnz; }
    }
    if ((int)blockIdx.x >= P.tile_prefix[P.n_clusters]) return;
    if (P.uniform_tiles > 0) {
      slot = (int)blockIdx.x / P.uniform_tiles;
    } else {
      int lo = 0, hi = P.n_clusters;
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (P.tile_prefix[mid] <= (int)blockIdx.x) lo = mid; else hi = mid;
      }
      slot = lo;
    }
    tile = __ldg(M.cluster_tile_begin + P.cluster[slot]) + ((int)blockIdx.x - P.tile_prefix[slot]);
  }
  TileDesc td;
  {
    const int4* src = reinterpret_cast<const int4*>(M.tiles + tile);
    int4* dst = reinterpret_cast<int4*>(&td);
#pragma unroll
    for (int i = 0; i < (int)(sizeof(TileDesc) / 16); ++i) dst[i] = __ldg(src + i);
  }
  const int nrows = td.nrows, t_lo = td.t_lo, s_int = td.s_int, s_ext = td.s_ext, nlo = td.nlo;
  const int S = s_int + s_ext;
  const int WT = C.WT, WV = C.WV;
#if GALE_CHECK_BOUNDS
  {
    bool ok = nrows >= 0 && nrows <= C.tv && NT >= 2 * C.tv && S >= 0 && S <= C.smax && s_ext <= C.sext &&
              td.nloc <= C.nloc && nlo >= 0 && nlo + nrows <= td.nloc && ((S + 31) >> 5) <= WT;
    if (mask & REL_VV) ok = ok && ((td.nloc + 31) >> 5) <= WV;
    if (!COUNT && (mask & REL_TT)) ok = ok && s_int <= C.sint && C.hs >= 2;
    if (!COUNT && (mask & (REL_VT | REL_TT))) ok = ok && td.vt_nnz <= C.vt_max;
    if (!COUNT && (mask & REL_VV)) ok = ok && td.vv_nnz <= C.vv_max;
    if (!ok) {  // block-uniform: leave before anything is staged
      if (tid == 0) raise_err(M.err, ERR_BOUNDS);
      return;
    }
  }
#endif

  unsigned char* tets = smem + L.tets;
  int32_t* texid = reinterpret_cast<int32_t*>(smem + L.texid);
  int32_t* gid = reinterpret_cast<int32_t*>(smem + L.gid);
  const int2* hft = reinterpret_cast<const int2*>(smem + L.hft);
  uint16_t* cnt = reinterpret_cast<uint16_t*>(smem + L.cnt);    // [2][tv] set bits of the row halves
  uint16_t* fbq = reinterpret_cast<uint16_t*>(smem + L.fbq);
  uint32_t* scan = reinterpret_cast<uint32_t*>(smem + L.scan);  // [0..33) scans, [36] queue length, [38] n_vv
  uint32_t* bmT = reinterpret_cast<uint32_t*>(smem + L.bmT);
  uint32_t* bmV = reinterpret_cast<uint32_t*>(smem + L.bmV);
  uint32_t* tbl = reinterpret_cast<uint32_t*>(smem + L.tbl);
  uint16_t* ttrow = reinterpret_cast<uint16_t*>(smem + L.ttrow);
  uint16_t* st_vt = reinterpret_cast<uint16_t*>(smem + L.st_vt);
  uint16_t* st_vv = reinterpret_cast<uint16_t*>(smem + L.st_vv);

  const int row0 = P.row_base[slot] + td.row_rel;
  const int vt0 = P.vt_base[slot] + td.vt_rel;
  const int vv0 = P.vv_base[slot] + td.vv_rel;
  const int tt0 = P.tt_base[slot] + td.tt_rel;

  // ---- P0: stage + clear ----------------------------------------------------------------------
  {
    const int4* src = reinterpret_cast<const int4*>(static_cast<const unsigned char*>(M.loc) + td.stg_off * (4 * LB));
    int4* dst = reinterpret_cast<int4*>(tets);
    for (int i = tid; i < (S * 4 * LB + 15) >> 4; i += NT) cp_async16(dst + i, src + i);
    {
      const int4* hsrc = reinterpret_cast<const int4*>(M.hft + td.gid_off);
      int4* hdst = reinterpret_cast<int4*>(smem + L.hft);
      for (int i = tid; i < (td.nloc + 1) >> 1; i += NT) cp_async16(hdst + i, hsrc + i);
    }
    if (!COUNT) {
      const int4* tsrc = reinterpret_cast<const int4*>(M.tex + td.tex_off);
      int4* tdst = reinterpret_cast<int4*>(texid);
      for (int i = tid; i < (s_ext + 3) >> 2; i += NT) cp_async16(tdst + i, tsrc + i);
      if (do_vv || do_tt) {
        const int4* gsrc = reinterpret_cast<const int4*>(M.gid + td.gid_off);
        int4* gdst = reinterpret_cast<int4*>(gid);
        for (int i = tid; i < (td.nloc + 3) >> 2; i += NT) cp_async16(gdst + i, gsrc + i);
      }
    }
  }
  {
    int4* z = reinterpret_cast<int4*>(smem + L.bmT);
    const int n16 = (L.bm_end - L.bmT) >> 4;
    for (int i = tid; i < n16; i += NT) z[i] = make_int4(0, 0, 0, 0);
  }
  if (do_tt) {  // tables empty, TT rows "none": both all-ones, contiguous
    int4* z = reinterpret_cast<int4*>(smem + L.tbl);
    const int n16 = (L.tt_end - L.tbl) >> 4;
    for (int i = tid; i < n16; i += NT) z[i] = make_int4(-1, -1, -1, -1);
  }
  if (tid == 0) { scan[36] = 0u; scan[38] = 0u; }
  cp_async_wait_all();
  __syncthreads();

  // ---- P1: VT incidence bits (rows = tile vertices, columns = staged simplices) ---------------
  for (int s = tid; s < S; s += NT) {
    int l[4];
    load_local<LB>(tets, s, l);
#if GALE_CHECK_BOUNDS
    for (int k = 0; k < D; ++k)
      if (!GALE_IN_BOUNDS(M.err, l[k] >= 0 && l[k] < td.nloc)) l[k] = nlo;  // keep later indexing inside the row
    if (s >= s_ext) (void)GALE_IN_BOUNDS(M.err, (unsigned)(l[0] - nlo) < (unsigned)nrows);  // internal: lowest vertex in the tile
#endif
    uint32_t* col = bmT + (s >> 5);
    const uint32_t bit = bit_of(s);
#pragma unroll
    for (int k = 1; k < D; ++k) {
      const int r = l[k] - nlo;
      if ((unsigned)r < (unsigned)nrows) atomicOr(col + r * WT, bit);
    }
    if (do_tt && s >= s_ext && l[1] - nlo >= nrows) {
      // facet 0 of this internal simplex leaves the tile (a5): its coface is almost always in the run
      // of the second vertex; pull those rows of T towards L2 now, they are read in the last phase
      const int2 run = hft[l[1]];
      const char* r0 = reinterpret_cast<const char*>(M.T) + (long long)run.x * (D * 4);
      const char* r1 = reinterpret_cast<const char*>(M.T) + (long long)max(run.y - 1, run.x) * (D * 4);
      asm volatile("prefetch.global.L2 [%0];" ::"l"(r0));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(r1));
    }
  }
  __syncthreads();

  // ---- P2: row degrees -> VT offsets ----------------------------------------------------------
  const bool isB = tid >= TV;
  const int p = isB ? tid - TV : tid;
  const bool live = p < nrows;
  const int ploc = nlo + p;
  const int wT = (S + 31) >> 5;
  if (live) {
    const int half = (wT + 1) >> 1;
    const uint32_t* row = bmT + p * WT;
    int c = 0;
    const int w0 = isB ? half : 0, w1 = isB ? wT : half;
#pragma unroll 4
    for (int w = w0; w < w1; ++w) c += __popc(row[w]);
    cnt[(isB ? C.tv : 0) + p] = (uint16_t)c;
  }
  __syncthreads();
  int nb = 0, off = 0, n_vt;
  {
    uint32_t deg = 0u, tot;
    if (live) {
      nb = (int)cnt[p] + (int)cnt[C.tv + p];
      const int2 run = hft[ploc];
      deg = (uint32_t)(nb + run.y - run.x);
    }
    const uint32_t ex = block_exclusive_scan<NT>(deg, scan, &tot);  // A and B halves carry the same values
    n_vt = (int)(tot >> 1);
    off = (int)ex - (isB ? n_vt : 0);
  }
  if (!COUNT && do_vt && live && !isB) O.vt_offsets[row0 + p] = vt0 + off;

  // ---- P3: A walks the bits of row p, B walks the run of p ------------------------------------
  if (live) {
    uint32_t* vvrow = bmV + p * WV;
    if (!isB) {
      const uint32_t* row = bmT + p * WT;
      int pos = off, sbase = -32;
      uint32_t bits = 0u;
      for (int n = 0; n < nb; ++n) {
        while (bits == 0u) { bits = *row++; sbase += 32; }
        const int s = sbase + __ffs(bits) - 1;
        bits &= bits - 1;
        int l[4];
        load_local<LB>(tets, s, l);
        if (entries && GALE_IN_BOUNDS(M.err, pos >= 0 && pos < C.vt_max && s >= 0 && s < S))
          st_vt[pos++] = (uint16_t)(s | (l[1] == ploc ? 0x8000 : 0));
        if (do_vv) {
#pragma unroll
          for (int k = 0; k < D; ++k) atomicOr(vvrow + (l[k] >> 5), bit_of(l[k]));  // self bit cleared in P4
        }
      }
    } else {
      GroupCtx g;
      if (do_tt) {
        const int hs = C.hs;
        g.tbl = tbl + p * (hs + 1);
        g.hs = (uint32_t)hs;
        g.ttrow = ttrow;
        g.s_ext = s_ext; g.s_all = S;
      }
      int pos = off + nb;
      const int2 run = hft[ploc];
      const int r1 = run.y - t_lo;
      for (int i = run.x - t_lo; i < r1; ++i) {
        const int s = s_ext + i;
        int l[4];
        load_local<LB>(tets, s, l);
        if (entries && GALE_IN_BOUNDS(M.err, pos >= 0 && pos < C.vt_max && s >= s_ext && s < S)) st_vt[pos++] = (uint16_t)s;
        if (do_vv) {
#pragma unroll
          for (int k = 1; k < D; ++k) atomicOr(vvrow + (l[k] >> 5), bit_of(l[k]));
        }
        if (do_tt) {
          group_place<D>(g, group_key<D, 1>(l), s, 1, M.err);
          group_place<D>(g, group_key<D, 2>(l), s, 2, M.err);
          if constexpr (D == 4) group_place<D>(g, group_key<D, 3>(l), s, 3, M.err);
        }
      }
    }
  }
  __syncthreads();

  // ---- P4: A joins the facets 0 of the simplices (x, p, ..); B expands VV row p ----------------
  int n_vv = 0;
  if (!isB) {
    if (do_tt && live) {
      GroupCtx g;
      const int hs = C.hs;
      g.tbl = tbl + p * (hs + 1);
      g.hs = (uint32_t)hs;
      g.ttrow = ttrow;
      g.s_ext = s_ext; g.s_all = S;
      int i = off;
      const int end = off + nb;
      for (;;) {
        uint32_t e = 0u;
        while (i < end && !((e = st_vt[i]) & 0x8000u)) ++i;
        if (i >= end) break;
        ++i;
        const int s = (int)(e & 0x7FFFu);
        int l[4];
        load_local<LB>(tets, s, l);
        group_place<D>(g, group_key<D, 0>(l), s, 0, M.err);
      }
    }
  } else if (do_vv) {
    const int wV = (td.nloc + 31) >> 5;
    uint32_t* row = bmV + p * WV;
    int nbv = 0;
    if (live) {
      row[ploc >> 5] &= ~bit_of(ploc);  // a vertex is not its own neighbour
#pragma unroll 4
      for (int w = 0; w < wV; ++w) nbv += __popc(row[w]);
    }
    uint32_t tot;
    const int offv = (int)half_exclusive_scan<NT>((uint32_t)nbv, scan, &tot);
    if (tid == TV) scan[38] = tot;
    if (live && !COUNT) {
      O.vv_offsets[row0 + p] = vv0 + offv;
      int pos = offv, lbase = -32;
      uint32_t bits = 0u;
      for (int n = 0; n < nbv; ++n) {
        while (bits == 0u) { bits = *row++; lbase += 32; }
        if (GALE_IN_BOUNDS(M.err, pos >= 0 && pos < C.vv_max && lbase + __ffs(bits) - 1 < td.nloc))
          st_vv[pos++] = (uint16_t)(lbase + __ffs(bits) - 1);
        bits &= bits - 1;
      }
    }
  }
  __syncthreads();
  n_vv = (int)scan[38];

  if (COUNT) {
    if (tid == 0) {
      O.stats[(long long)tile * 4 + 0] = n_vt;
      O.stats[(long long)tile * 4 + 1] = n_vv;
      O.stats[(long long)tile * 4 + 2] = 0;
      O.stats[(long long)tile * 4 + 3] = 0;
    }
    return;
  }
  if (tid == 0 && ((do_vt && n_vt != td.vt_nnz) || (do_vv && n_vv != td.vv_nnz)))
    raise_err(M.err, ERR_SIZE_MISMATCH);  // the sizes fixed at create must be reproduced exactly

  // ---- P5: translate to global ids, coalesced write-out ----------------------------------------
  if (do_tt) {
    // facets no tile vertex owns go to the queue
    for (int base = tid - lane; base < s_int; base += NT) {  // warp-uniform trip count
      const int i = base + lane;
      bool need_fb = false;
      if (i < s_int) {
        uint32_t e[D];
        if constexpr (D == 4) {
          const uint2 q = reinterpret_cast<const uint2*>(ttrow)[i];
          e[0] = q.x & 0xFFFFu; e[1] = q.x >> 16; e[2] = q.y & 0xFFFFu; e[3] = q.y >> 16;
        } else {
          e[0] = ttrow[i * 3]; e[1] = ttrow[i * 3 + 1]; e[2] = ttrow[i * 3 + 2];
        }
        int r[D];
#pragma unroll
        for (int k = 0; k < D; ++k)
          r[k] = e[k] == 0xFFFFu ? -1 : ((int)e[k] < s_ext ? texid[e[k]] : t_lo + ((int)e[k] - s_ext));
        if constexpr (D == 4) {
          GALE_ST(reinterpret_cast<int4*>(O.tt_indices) + tt0 + i, make_int4(r[0], r[1], r[2], r[3]));
        } else {
          int32_t* o = O.tt_indices + (long long)(tt0 + i) * 3;
          o[0] = r[0]; o[1] = r[1]; o[2] = r[2];
        }
        if (r[0] < 0) {
          int l[4];
          load_local<LB>(tets, s_ext + i, l);
          need_fb = l[1] - nlo >= nrows;
        }
      }
      const unsigned fbm = __ballot_sync(0xFFFFFFFFu, need_fb);
      if (fbm) {
        const int leader = __ffs(fbm) - 1;
        uint32_t pos = 0u;
        if (lane == leader) pos = atomicAdd(&scan[36], (uint32_t)__popc(fbm));
        pos = __shfl_sync(0xFFFFFFFFu, pos, leader);
        if (need_fb && GALE_IN_BOUNDS(M.err, (int)(pos + __popc(fbm & ((1u << lane) - 1u))) < C.sint))
          fbq[pos + __popc(fbm & ((1u << lane) - 1u))] = (uint16_t)i;
      }
    }
  }
  if (do_vt)
    for (int i = tid; i < n_vt; i += NT) {
      const int s = (int)(st_vt[i] & 0x7FFFu);
      GALE_ST(O.vt_indices + vt0 + i, s < s_ext ? texid[s] : t_lo + (s - s_ext));
    }
  if (do_vv)
    for (int i = tid; i < n_vv; i += NT) GALE_ST(O.vv_indices + vv0 + i, gid[st_vv[i]]);

  if (do_tt) {
    __syncthreads();  // queue complete, TT rows stored
    // ---- a5: one queued facet per thread, resolved from global memory -------------------------
    const int nq = (int)scan[36];
    for (int q = tid; q < nq; q += NT) {
      const int i = fbq[q];
      int l[4];
      load_local<LB>(tets, s_ext + i, l);
      const int t = t_lo + i;
      const int b = gid[l[1]], c = gid[l[2]], d = D == 4 ? gid[l[3]] : 0;
      const int2 run = hft[l[1]];
      const int r = tt_fallback<D>(M, run.x, run.y, b, c, d, t);
      if (r >= 0) O.tt_indices[(long long)(tt0 + i) * D] = r;  // ordered after the row store by the barrier
    }
  }
}

}  // namespace gale
