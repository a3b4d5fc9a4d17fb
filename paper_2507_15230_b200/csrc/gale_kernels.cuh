// gale_kernels.cuh — sm_100a kernels of the GALE relation hot path.
//
// One thread block owns one *tile*: a contiguous vertex sub-range [v_lo, v_lo+nrows) of a cluster
// (a tile plays the role of the paper's <=100-vertex segment; a cluster is the
// request unit). gale_mesh_create stores, per tile, the simplices incident to it
// (internal ones = rows I_T of T; external ones = the tile's T_ex list)
// re-encoded in *tile-local* 16-bit vertex ids that ascend with the global id:
//     [lower halo 0..nlo) [tile vertices nlo..nlo+nrows) [upper halo ..nloc)
// ("halo" = vertices outside the tile that share a simplex with it), external simplices first.
// Every external simplex has a smaller global id than every internal one (its lowest vertex lies
// below the tile), so the staged order s = 0..S-1 ascends with the global simplex id.
//
// Phases of a block:
//   a1  stage the list (8 B per simplex), the external simplices' global ids, the local->global
//       vertex table and the tile's second-vertex index into shared memory with 16-byte cp.async;
//   a4  TT, one thread per tile vertex p and no atomics: a facet whose lowest vertex is p has all
//       its cofaces among the simplices whose lowest vertex is p (the contiguous run
//       first_tet[p]..first_tet[p+1], facets 1..D-1) and the staged simplices whose second vertex
//       is p (their facet 0; listed per tile vertex by the create-time index, like the paper's
//       sorted lists bounded by interval arrays). The thread walks these
//       few records through a private open-addressing table keyed by the facet's other vertices;
//       the second arrival of a key meets the first and both TT entries are written to a
//       shared-memory copy of the tile's TT rows;
//   a5  TT fallback: the facet opposite the lowest vertex a of an internal simplex (a,b,..) with b
//       outside the tile belongs to no vertex of the tile; such facets are compacted into a queue
//       and resolved one per thread from global memory through the run of simplices starting with
//       b and the index of simplices whose second vertex is b (DESIGN.md §TT fallback);
//   a2  VT: one bit per (row, staged simplex) in a rows x S bitmap (atomicOr); expanding a row
//       yields its simplices in ascending order with no sort; the simplices whose *lowest* vertex
//       is v are the contiguous run first_tet[v]..first_tet[v+1] and are appended without bits;
//   a3  VV: one bit per (row, local neighbour) in a rows x nloc bitmap (atomicOr: "no duplicates",
//       PAPER.md:228); local ids ascend with global ids, so a row expands sorted;
//   a6  rows are expanded into shared-memory staging (ids translated back to global) and written
//       out with coalesced stores.
// All arithmetic is integer index work; no floating point.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gale {

constexpr int kMaxBatch = 128;         // clusters per kernel launch (descriptor lives in kernel params)
constexpr uint32_t kEmpty32 = 0xFFFFFFFFu;
constexpr int kMaxStaged = 65534;      // staged simplices per tile (16-bit staged indices)
constexpr int kMaxLocal4 = 1024;       // tetrahedra: 10-bit local ids (20-bit facet key + 12-bit record)
constexpr int kMaxLocal3 = 65534;      // triangles: 16-bit local ids (16-bit facet key + 16-bit record)
constexpr int kMaxGroup4 = 4095;       // facet records of one vertex (tetrahedra / triangles)
constexpr int kMaxGroup3 = 65534;
constexpr int kMaxNnz16 = 65535;       // VT / VV entries of one tile (16-bit packed scan)

enum { REL_VT = 1, REL_VV = 2, REL_TT = 4, MODE_COUNT = 8 };
enum { ERR_TT_TABLE_FULL = 2, ERR_SIZE_MISMATCH = 4 };

// Per-tile record built by gale_mesh_create (96 bytes, 16-byte aligned).
struct TileDesc {
  int32_t v_lo, nrows;        // vertices [v_lo, v_lo+nrows)
  int32_t t_lo, s_int;        // internal simplices [t_lo, t_lo+s_int)
  int32_t s_ext;              // external simplices (T_ex of the tile)
  int32_t nlo, nloc;          // halo vertices below v_lo / local ids in total (halo + rows)
  int32_t row_rel, tt_rel;    // first row / first TT row of the tile inside its cluster
  int32_t vt_rel, vv_rel;     // first VT / VV entry of the tile inside its cluster
  int32_t vt_nnz, vv_nnz;     // entries of the tile (fixed at create; the kernel re-derives them)
  int32_t n_opp;              // staged simplices whose second vertex is in the tile
  long long stg_off;          // first staged simplex of the tile in DeviceMesh::loc (even)
  long long tex_off;          // first entry in DeviceMesh::tex (multiple of 4)
  long long gid_off;          // first entry in DeviceMesh::gid (multiple of 4)
  long long opp_off;          // first entry in DeviceMesh::opp (multiple of 8)
  long long pad0;
};
static_assert(sizeof(TileDesc) == 96, "TileDesc layout");

// Device-resident index built by gale_mesh_create (all pointers DEVICE).
struct DeviceMesh {
  const int32_t* T;                   // [nT*D] canonical simplices (caller's array)
  const int32_t* first_tet;           // [nV+1] first simplex whose lowest vertex is >= v  (I_T)
  const int32_t* opp_first;           // [nV+1] first position in opp_perm whose second vertex is >= v
  const int32_t* opp_perm;            // [nT]   simplex ids grouped by second vertex
  const TileDesc* tiles;              // [nTiles]
  const uint2* loc;                   // staged simplices in tile-local ids, 4 x uint16 each
  const int32_t* tex;                 // per-tile ascending global ids of external simplices (T_ex)
  const int32_t* gid;                 // per-tile global vertex id of every local id (ascending)
  const uint16_t* opp;                // per tile: [tv_pad] start of row r, then the staged indices of the
                                      // simplices whose second vertex is row r, ascending, rows in order
  const int32_t* cluster_tile_begin;  // [nC+1]
  int32_t* err;                       // sticky device error flags (host-mapped)
};

// Shared-memory capacities (maxima over all tiles of the mesh, fixed at create). A field is 0 when
// the launch's relation mask does not need the region.
struct SmemCfg {
  int tv;        // rows (vertices) per tile, <= NT/2
  int smax;      // staged simplices (even)
  int sext;      // external simplices (multiple of 4)
  int nloc;      // local vertex ids (multiple of 4)
  int sint;      // internal simplices (even): TT row copy + fallback queue, 0 without TT
  int nopp;      // second-vertex index entries incl. the row starts (multiple of 8), 0 without TT
  int hs;        // table slots per tile vertex (power of two), 0 without TT
  int WT;        // VT bitmap words per row (odd), 0 without VT
  int WV;        // VV bitmap words per row (odd), 0 without VV
  int vt_max;    // VT entries staged for write-out, 0 without VT or in count mode
  int vv_max;    // VV entries staged for write-out
};

// Byte offsets of the shared-memory regions, computed on the host (make_layout) and passed as a
// kernel parameter. The TT tables / TT row copy and the VT/VV staging share one union (the tables
// are dead before the rows are expanded).
struct SmemLayout {
  int tets, texid, gid, opp, ft, off_vt, off_vv, fbq, scan, bmT, bmV, bm_end;
  int tbl, ttrow, tt_end;           // TT phase
  int st_vt, st_vv;                 // write-out staging
  int total;
};

__host__ __device__ inline int align16(int x) { return (x + 15) & ~15; }
__host__ __device__ inline int opp_rows_pad(int tv) { return (tv + 1 + 7) & ~7; }

template <int D>
__host__ __device__ inline SmemLayout make_layout(const SmemCfg& c) {
  SmemLayout L;
  int o = 0;
  L.tets = o;   o = align16(o + c.smax * 8);
  L.texid = o;  o = align16(o + c.sext * 4);
  L.gid = o;    o = align16(o + c.nloc * 4);
  L.opp = o;    o = align16(o + c.nopp * 2);
  L.ft = o;     o = align16(o + (c.tv + 1) * 4);
  L.off_vt = o; o = align16(o + (c.tv + 1) * 4);
  L.off_vv = o; o = align16(o + (c.tv + 1) * 4);
  L.fbq = o;    o = align16(o + c.sint * 2);
  L.scan = o;   o = align16(o + 48 * 4);
  L.bmT = o;    o = align16(o + c.tv * c.WT * 4);
  L.bmV = o;    o = align16(o + c.tv * c.WV * 4);
  L.bm_end = o;
  L.tbl = o;    o = align16(o + (c.hs ? c.tv * (c.hs + 1) * 4 : 0));
  L.ttrow = o;  o = align16(o + c.sint * D * 4);
  L.tt_end = o;
  o = L.tbl;
  L.st_vt = o;  o = align16(o + c.vt_max * 4);
  L.st_vv = o;  o = align16(o + c.vv_max * 4);
  L.total = o > L.tt_end ? o : L.tt_end;
  return L;
}

// Per-launch batch descriptor, passed by value in kernel parameter space (no H2D copy).
struct BatchParams {
  int n_clusters;
  uint32_t mask;
  int tile_base;                     // count mode: first tile of the launch
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
  long long* stats;                  // count mode: [nTiles][4] = VT nnz, VV nnz, 0, 0
};

// ------------------------------------------------------------------------------------------------
// Guard codes go to a host-mapped word (plain store: no PCIe atomics needed; any code is fatal).
__device__ __forceinline__ void raise_err(int32_t* err, int code) { *reinterpret_cast<volatile int32_t*>(err) = code; }

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

__device__ __forceinline__ void unpack_local(const uint2 q, int (&l)[4]) {
  l[0] = q.x & 0xFFFF; l[1] = q.x >> 16; l[2] = q.y & 0xFFFF; l[3] = q.y >> 16;
}

template <int D>
__device__ __forceinline__ void load_simplex_global(const int32_t* T, int t, int (&v)[4]) {
  if constexpr (D == 4) {
    const int4 q = __ldg(reinterpret_cast<const int4*>(T) + t);
    v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
  } else {
    v[0] = __ldg(T + (long long)t * 3); v[1] = __ldg(T + (long long)t * 3 + 1); v[2] = __ldg(T + (long long)t * 3 + 2);
    v[3] = -1;
  }
}

// a5, one request per thread: coface != self of the facet (b, c[, d]) (ascending global ids) whose
// vertices all lie outside the tile. Both cofaces of a facet with lowest vertex b have b as
// lowest or second-lowest vertex: candidates are the run of simplices starting with b (sorted, so
// the scan stops once the second vertex exceeds c) and the simplices whose second vertex is b
// (those are (x, b, c, d) exactly).
template <int D>
__device__ __forceinline__ int tt_fallback(const DeviceMesh& M, int b, int c, int d, int self) {
  const int f0 = __ldg(M.first_tet + b), f1 = __ldg(M.first_tet + b + 1);
  const int o0 = __ldg(M.opp_first + b), o1 = __ldg(M.opp_first + b + 1);
  for (int t = f0; t < f1; ++t) {
    int v[4];
    load_simplex_global<D>(M.T, t, v);
    if (v[1] > c) break;
    bool hit;
    if constexpr (D == 4) hit = (v[1] == c && (v[2] == d || v[3] == d)) || (v[2] == c && v[3] == d);
    else hit = v[1] == c || v[2] == c;
    if (hit) return t;
  }
  for (int j = o0; j < o1; ++j) {
    const int t = __ldg(M.opp_perm + j);
    if (t == self) continue;
    int v[4];
    load_simplex_global<D>(M.T, t, v);
    bool hit;
    if constexpr (D == 4) hit = v[2] == c && v[3] == d;
    else hit = v[2] == c;
    if (hit) return t;
  }
  return -1;
}

// Block-wide exclusive scan of one value per thread. Returns the exclusive prefix; *total gets
// the block sum. scratch: 33 ints of shared memory.
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
// a4 helpers. A facet record of vertex p's group is numbered j: first the facets 1..D-1 of the
// simplices of the run of p (j = (D-1) * q + k-1 for the q-th simplex of the run), then facet 0 of
// the simplices whose second vertex is p, in the order of the tile's second-vertex index.
template <int D>
struct FacetBits {  // table word = key | (j << kKeyBits); the key holds the facet's vertices other than p
  static constexpr int kKeyBits = D == 4 ? 20 : 16;
  static constexpr uint32_t kKeyMask = (1u << kKeyBits) - 1u;
};

struct GroupCtx {
  uint32_t* tbl;           // this vertex's table, hs slots
  uint32_t hmask;
  int hshift;
  int32_t* ttrow;          // shared-memory copy of the tile's TT rows, D entries per internal simplex
  const int32_t* texid;
  const uint16_t* opp_idx; // second-vertex records of p
  int run0;                // first internal simplex (index in the tile) of the run of p
  int nrun;                // (D-1) * simplices in the run
  int s_ext, t_lo;
};

__device__ __forceinline__ int global_simplex(const GroupCtx& g, int s) {
  return s < g.s_ext ? g.texid[s] : g.t_lo + (s - g.s_ext);
}

// Place record j = facet k of staged simplex s with key `key`: claim an empty slot, or meet the
// record that holds the same key (the other coface) and write both TT entries.
template <int D>
__device__ __forceinline__ void group_place(const GroupCtx& g, uint32_t key, int j, int s, int k, int32_t* err) {
  using FB = FacetBits<D>;
  uint32_t h = (key * 0x9E3779B1u) >> g.hshift;
  for (uint32_t probe = 0; probe <= g.hmask; ++probe) {
    const uint32_t cur = g.tbl[h];
    if (cur == kEmpty32) {
      g.tbl[h] = key | ((uint32_t)j << FB::kKeyBits);
      return;
    }
    if ((cur & FB::kKeyMask) == key) {
      const int j2 = (int)(cur >> FB::kKeyBits);
      int s2, k2;
      if (j2 < g.nrun) {
        const int q = j2 / (D - 1);
        s2 = g.s_ext + g.run0 + q;
        k2 = 1 + j2 - q * (D - 1);
      } else {
        s2 = g.opp_idx[j2 - g.nrun];
        k2 = 0;
      }
      if (s >= g.s_ext) g.ttrow[(s - g.s_ext) * D + k] = global_simplex(g, s2);
      if (s2 >= g.s_ext) g.ttrow[(s2 - g.s_ext) * D + k2] = global_simplex(g, s);
      return;
    }
    h = (h + 1) & g.hmask;
  }
  raise_err(err, ERR_TT_TABLE_FULL);
}

// Key of the facet of a simplex with lowest vertex p that omits local vertex K (1 <= K < D): the
// facet's vertices other than p, ascending. For K = 0 (simplex (x, p, ..)): the vertices after p.
template <int D, int K>
__device__ __forceinline__ uint32_t group_key(const int (&l)[4]) {
  if constexpr (D == 4) {
    const int a = K <= 1 ? l[2] : l[1];
    const int b = (K == 0 || K == 1 || K == 2) ? l[3] : l[2];
    return (uint32_t)a | ((uint32_t)b << 10);
  } else {
    return (uint32_t)(K <= 1 ? l[2] : l[1]);
  }
}

// ------------------------------------------------------------------------------------------------
// The batch kernel: VT + VV + TT for every tile of the requested clusters (or, COUNT, the exact
// VT / VV sizes of tiles [tile_base, tile_base + gridDim.x) — the paper's leader producer likewise
// sizes its relation arrays before launch). NT >= 2 * rows per tile.
template <int D, int NT, bool COUNT>
__global__ void __launch_bounds__(NT, (NT <= 128 ? 8 : (NT <= 256 ? 4 : 2)))
gale_batch_kernel(const DeviceMesh M, const __grid_constant__ BatchParams P, const SmemCfg C,
                  const SmemLayout L, const OutPtrs O) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x, lane = tid & 31;
  const uint32_t mask = P.mask;
  const bool do_vt = (mask & REL_VT) != 0, do_vv = (mask & REL_VV) != 0;
  const bool do_tt = !COUNT && (mask & REL_TT) != 0;

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
    int lo = 0, hi = P.n_clusters;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (P.tile_prefix[mid] <= (int)blockIdx.x) lo = mid; else hi = mid;
    }
    slot = lo;
    tile = __ldg(M.cluster_tile_begin + P.cluster[slot]) + ((int)blockIdx.x - P.tile_prefix[slot]);
  }
  TileDesc td;
  {
    const int4* src = reinterpret_cast<const int4*>(M.tiles + tile);
    int4* dst = reinterpret_cast<int4*>(&td);
#pragma unroll
    for (int i = 0; i < (int)(sizeof(TileDesc) / 16); ++i) dst[i] = __ldg(src + i);
  }
  const int v_lo = td.v_lo, nrows = td.nrows, t_lo = td.t_lo, s_int = td.s_int, s_ext = td.s_ext, nlo = td.nlo;
  const int S = s_int + s_ext;
  const int WT = C.WT, WV = C.WV;

  uint2* tets = reinterpret_cast<uint2*>(smem + L.tets);
  int32_t* texid = reinterpret_cast<int32_t*>(smem + L.texid);
  int32_t* gid = reinterpret_cast<int32_t*>(smem + L.gid);
  uint16_t* opp = reinterpret_cast<uint16_t*>(smem + L.opp);
  int32_t* ft = reinterpret_cast<int32_t*>(smem + L.ft);
  int32_t* off_vt = reinterpret_cast<int32_t*>(smem + L.off_vt);
  int32_t* off_vv = reinterpret_cast<int32_t*>(smem + L.off_vv);
  uint16_t* fbq = reinterpret_cast<uint16_t*>(smem + L.fbq);
  uint32_t* scan = reinterpret_cast<uint32_t*>(smem + L.scan);  // [0..33) scan, [36] queue length, [37] chunk counter
  uint32_t* bmT = reinterpret_cast<uint32_t*>(smem + L.bmT);
  uint32_t* bmV = reinterpret_cast<uint32_t*>(smem + L.bmV);
  uint32_t* tbl = reinterpret_cast<uint32_t*>(smem + L.tbl);
  int32_t* ttrow = reinterpret_cast<int32_t*>(smem + L.ttrow);
  int32_t* st_vt = reinterpret_cast<int32_t*>(smem + L.st_vt);
  int32_t* st_vv = reinterpret_cast<int32_t*>(smem + L.st_vv);

  const int row0 = P.row_base[slot] + td.row_rel;
  const int vt0 = P.vt_base[slot] + td.vt_rel;
  const int vv0 = P.vv_base[slot] + td.vv_rel;
  const int tt0 = P.tt_base[slot] + td.tt_rel;
  const int opp_rows = opp_rows_pad(nrows);

  // ---- a1: stage + clear ----------------------------------------------------------------------
  {
    const int4* src = reinterpret_cast<const int4*>(M.loc + td.stg_off);
    int4* dst = reinterpret_cast<int4*>(tets);
    for (int i = tid; i < (S + 1) >> 1; i += NT) cp_async16(dst + i, src + i);
    const int4* tsrc = reinterpret_cast<const int4*>(M.tex + td.tex_off);
    int4* tdst = reinterpret_cast<int4*>(texid);
    for (int i = tid; i < (s_ext + 3) >> 2; i += NT) cp_async16(tdst + i, tsrc + i);
    const int4* gsrc = reinterpret_cast<const int4*>(M.gid + td.gid_off);
    int4* gdst = reinterpret_cast<int4*>(gid);
    for (int i = tid; i < (td.nloc + 3) >> 2; i += NT) cp_async16(gdst + i, gsrc + i);
    if (do_tt) {
      const int4* osrc = reinterpret_cast<const int4*>(M.opp + td.opp_off);
      int4* odst = reinterpret_cast<int4*>(opp);
      for (int i = tid; i < (opp_rows + td.n_opp + 7) >> 3; i += NT) cp_async16(odst + i, osrc + i);
    }
  }
  for (int i = tid; i <= nrows; i += NT) ft[i] = __ldg(M.first_tet + v_lo + i) - t_lo;
  {
    int4* z = reinterpret_cast<int4*>(smem + L.bmT);
    const int n16 = (L.bm_end - L.bmT) >> 4;
    for (int i = tid; i < n16; i += NT) z[i] = make_int4(0, 0, 0, 0);
  }
  if (do_tt) {  // tables empty, TT rows -1: both all-ones, contiguous
    int4* z = reinterpret_cast<int4*>(smem + L.tbl);
    const int n16 = (L.tt_end - L.tbl) >> 4;
    for (int i = tid; i < n16; i += NT) z[i] = make_int4(-1, -1, -1, -1);
  }
  if (tid < 2) scan[36 + tid] = 0u;
  cp_async_wait_all();
  __syncthreads();

  // ---- a4: thread p matches the facets whose lowest vertex is tile vertex p -------------------
  if (do_tt && tid < nrows) {
    GroupCtx g;
    const int hs = C.hs;
    g.tbl = tbl + tid * (hs + 1);
    g.hmask = (uint32_t)hs - 1u;
    g.hshift = 32 - (31 - __clz(hs));
    g.ttrow = ttrow;
    g.texid = texid;
    const int r0 = ft[tid], r1 = ft[tid + 1];
    const int o0 = opp[tid], o1 = opp[tid + 1];
    g.opp_idx = opp + opp_rows + o0;
    g.run0 = r0;
    g.nrun = (r1 - r0) * (D - 1);
    g.s_ext = s_ext;
    g.t_lo = t_lo;
    int j = 0;
    for (int i = r0; i < r1; ++i) {
      int l[4];
      unpack_local(tets[s_ext + i], l);
      group_place<D>(g, group_key<D, 1>(l), j, s_ext + i, 1, M.err);
      group_place<D>(g, group_key<D, 2>(l), j + 1, s_ext + i, 2, M.err);
      if constexpr (D == 4) group_place<D>(g, group_key<D, 3>(l), j + 2, s_ext + i, 3, M.err);
      j += D - 1;
    }
    for (int o = o0; o < o1; ++o, ++j) {
      const int s = opp[opp_rows + o];
      int l[4];
      unpack_local(tets[s], l);
      group_place<D>(g, group_key<D, 0>(l), j, s, 0, M.err);
    }
  }

  // ---- a2/a3: one bit per incidence / per adjacent pair; warps take chunks of 32 simplices -----
  if (do_vt || do_vv) {
    const int nchunks = (S + 31) >> 5;
    for (;;) {
      uint32_t c = 0u;
      if (lane == 0) c = atomicAdd(&scan[37], 1u);
      c = __shfl_sync(0xFFFFFFFFu, c, 0);
      if ((int)c >= nchunks) break;
      const int s = (int)c * 32 + lane;
      if (s < S) {
        int l[4];
        unpack_local(tets[s], l);
        bool in[D];
#pragma unroll
        for (int k = 0; k < D; ++k) in[k] = (unsigned)(l[k] - nlo) < (unsigned)nrows;
        if (do_vt) {
          const uint32_t bit = 1u << lane;
          uint32_t* col = bmT + c;
#pragma unroll
          for (int k = 1; k < D; ++k)
            if (in[k]) atomicOr(col + (l[k] - nlo) * WT, bit);
        }
        if (do_vv) {
          uint32_t w[D], b[D];
#pragma unroll
          for (int k = 0; k < D; ++k) { w[k] = (uint32_t)l[k] >> 5; b[k] = 1u << (l[k] & 31); }
#pragma unroll
          for (int k = 0; k < D; ++k) {
            if (!in[k]) continue;
            uint32_t* row = bmV + (l[k] - nlo) * WV;
#pragma unroll
            for (int j = 0; j < D; ++j)
              if (j != k) atomicOr(row + w[j], b[j]);
          }
        }
      }
    }
  }
  __syncthreads();

  if (do_tt) {
    // ---- TT rows to global; facets no tile vertex owns go to the queue --------------------------
    for (int base = tid - lane; base < s_int; base += NT) {  // warp-uniform trip count
      const int i = base + lane;
      bool need_fb = false;
      if (i < s_int) {
        int first;
        if constexpr (D == 4) {
          const int4 v = reinterpret_cast<const int4*>(ttrow)[i];
          reinterpret_cast<int4*>(O.tt_indices)[tt0 + i] = v;
          first = v.x;
        } else {
          int32_t* o = O.tt_indices + (long long)(tt0 + i) * 3;
          first = ttrow[i * 3];
          o[0] = first; o[1] = ttrow[i * 3 + 1]; o[2] = ttrow[i * 3 + 2];
        }
        need_fb = first < 0 && (int)(tets[s_ext + i].x >> 16) - nlo >= nrows;
      }
      const unsigned fbm = __ballot_sync(0xFFFFFFFFu, need_fb);
      if (fbm) {
        const int leader = __ffs(fbm) - 1;
        uint32_t pos = 0u;
        if (lane == leader) pos = atomicAdd(&scan[36], (uint32_t)__popc(fbm));
        pos = __shfl_sync(0xFFFFFFFFu, pos, leader);
        if (need_fb) fbq[pos + __popc(fbm & ((1u << lane) - 1u))] = (uint16_t)i;
      }
    }
  }

  if (do_vt || do_vv) {
    // ---- row degrees -> offsets: threads [0, rows) own the VT rows, [NT/2, NT/2+rows) the VV rows
    const bool vt_thread = do_vt && tid < nrows;
    const int vrow = tid - NT / 2;
    const bool vv_thread = do_vv && vrow >= 0 && vrow < nrows;
    const int wT = (S + 31) >> 5, wV = (td.nloc + 31) >> 5;
    uint32_t tot = 0u;
    int nbits = 0;  // set bits of this thread's row
    {
      uint32_t deg = 0u;
      if (vt_thread) {
        const uint32_t* row = bmT + tid * WT;
#pragma unroll 4
        for (int w = 0; w < wT; ++w) nbits += __popc(row[w]);
        deg = (uint32_t)(nbits + ft[tid + 1] - ft[tid]);
      } else if (vv_thread) {
        const uint32_t* row = bmV + vrow * WV;
#pragma unroll 4
        for (int w = 0; w < wV; ++w) nbits += __popc(row[w]);
        deg = (uint32_t)nbits << 16;
      }
      const uint32_t ex = block_exclusive_scan<NT>(deg, scan, &tot);  // (also orders the TT row copy
      if (vt_thread) off_vt[tid] = (int)(ex & 0xFFFFu);               //  before the staging reuse)
      if (vv_thread) off_vv[vrow] = (int)(ex >> 16);
    }
    const int n_vt = (int)(tot & 0xFFFFu), n_vv = (int)(tot >> 16);
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

    // ---- expand the rows into the staging areas, ids translated back to global ------------------
    // One loop iteration per set bit (not per word): lanes of a warp run in step however their
    // bits are spread over the words of their rows.
    if (vt_thread) {
      O.vt_offsets[row0 + tid] = vt0 + (int)off_vt[tid];
      const uint32_t* row = bmT + tid * WT;
      int p = off_vt[tid], sbase = -32;
      uint32_t bits = 0u;
      for (int n = 0; n < nbits; ++n) {
        while (bits == 0u) { bits = *row++; sbase += 32; }
        const int s = sbase + __ffs(bits) - 1;
        bits &= bits - 1;
        st_vt[p++] = s < s_ext ? texid[s] : t_lo + (s - s_ext);
      }
      for (int j = ft[tid]; j < ft[tid + 1]; ++j) st_vt[p++] = t_lo + j;
    } else if (vv_thread) {
      O.vv_offsets[row0 + vrow] = vv0 + (int)off_vv[vrow];
      const uint32_t* row = bmV + vrow * WV;
      int p = off_vv[vrow], lbase = -32;
      uint32_t bits = 0u;
      for (int n = 0; n < nbits; ++n) {
        while (bits == 0u) { bits = *row++; lbase += 32; }
        const int l = lbase + __ffs(bits) - 1;
        bits &= bits - 1;
        st_vv[p++] = gid[l];
      }
    }
    __syncthreads();

    // ---- a6: coalesced write-out ----------------------------------------------------------------
    if (do_vt)
      for (int i = tid; i < n_vt; i += NT) O.vt_indices[vt0 + i] = st_vt[i];
    if (do_vv)
      for (int i = tid; i < n_vv; i += NT) O.vv_indices[vv0 + i] = st_vv[i];
  } else {
    __syncthreads();  // queue complete
  }

  if (do_tt) {
    // ---- a5: one queued facet per thread, resolved from global memory (no barrier follows) ------
    const int nq = (int)scan[36];
    for (int q = tid; q < nq; q += NT) {
      const int i = fbq[q];
      int l[4];
      unpack_local(tets[s_ext + i], l);
      const int b = gid[l[1]], c = gid[l[2]], d = D == 4 ? gid[l[3]] : 0;
      const int r = tt_fallback<D>(M, b, c, d, t_lo + i);
      if (r >= 0) O.tt_indices[(long long)(tt0 + i) * D] = r;  // ordered after the row store by the barriers
    }
  }
}

}  // namespace gale
